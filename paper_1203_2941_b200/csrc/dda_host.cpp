// dda_host.cpp -- host-side driver of csrc/dda.h for tests/test_dda_host.py (-m "not gpu").
// Walks a ray through a grid the way k_transport does -- cell by cell where a cell or its box holds dust,
// mcrt::box_jump over boxes of vacuum cells -- and reports what the transport needs to be identical to the
// plain cell-by-cell walk: the (cell, ds) list of the dusty cells, the number of faces crossed and the
// parameter of the exit face.  Compiled with g++ -ffp-contract=off; no physics, no oracle code.
#include <stdint.h>

#include <vector>

#include "dda.h"

namespace {

struct Masks {
    int msh, nx, ny, nz;
    int mb[3][3];
    std::vector<uint8_t> m[3];
    bool empty(int l, int ix, int iy, int iz) const
    {
        const int sh = msh + 2 * l;
        return m[l][((size_t)(iz >> sh) * mb[l][1] + (iy >> sh)) * mb[l][0] + (ix >> sh)] != 0;
    }
};

Masks build_masks(const uint8_t *dusty, int nx, int ny, int nz, int msh)
{
    Masks M;
    M.msh = msh; M.nx = nx; M.ny = ny; M.nz = nz;
    for (int l = 0; l < 3; ++l) {
        const int e = 1 << (msh + 2 * l);
        M.mb[l][0] = (nx + e - 1) / e; M.mb[l][1] = (ny + e - 1) / e; M.mb[l][2] = (nz + e - 1) / e;
        M.m[l].assign((size_t)M.mb[l][0] * M.mb[l][1] * M.mb[l][2], 1);
    }
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x)
                if (dusty[((size_t)z * ny + y) * nx + x])
                    for (int l = 0; l < 3; ++l) {
                        const int sh = msh + 2 * l;
                        M.m[l][((size_t)(z >> sh) * M.mb[l][1] + (y >> sh)) * M.mb[l][0] + (x >> sh)] = 0;
                    }
    return M;
}

}  // namespace

extern "C" {

// Returns the number of dusty cells listed (cells/ds_out hold at most max_n); *faces = all faces crossed,
// *t_exit = parameter of the last face, *jumps = number of box jumps taken.  c0 = start cell.
int mcrt_dda_host_trace(int nx, int ny, int nz, const uint8_t *dusty, int msh, const double p[3], const double u[3],
                        const int c0[3], int use_jumps, int max_n, int64_t *cells, double *ds_out, uint64_t *faces,
                        double *t_exit, int *jumps)
{
    const Masks M = build_masks(dusty, nx, ny, nz, msh);
    int ix = c0[0], iy = c0[1], iz = c0[2];
    const int stx = (u[0] > 0.0) ? 1 : ((u[0] < 0.0) ? -1 : 0);
    const int sty = (u[1] > 0.0) ? 1 : ((u[1] < 0.0) ? -1 : 0);
    const int stz = (u[2] > 0.0) ? 1 : ((u[2] < 0.0) ? -1 : 0);
    const double ivx = stx ? 1.0 / u[0] : (double)INFINITY;
    const double ivy = sty ? 1.0 / u[1] : (double)INFINITY;
    const double ivz = stz ? 1.0 / u[2] : (double)INFINITY;
    double tmx = mcrt::face_t(ix, stx, p[0], ivx), tmy = mcrt::face_t(iy, sty, p[1], ivy),
           tmz = mcrt::face_t(iz, stz, p[2], ivz);
    double t = 0.0;
    uint64_t nf = 0;
    int cnt = 0, nj = 0;
    for (;;) {
        if ((unsigned)ix >= (unsigned)nx || (unsigned)iy >= (unsigned)ny || (unsigned)iz >= (unsigned)nz) break;
        const bool d = dusty[((size_t)iz * ny + iy) * nx + ix] != 0;
        if (use_jumps == 2 && !d && M.empty(0, ix, iy, iz)) {
            // the kernel's box: cube of bricks closer (max norm) than the nearest brick with dust
            const int bx = ix >> msh, by = iy >> msh, bz = iz >> msh;
            int dd = 255;
            for (int z = 0; z < M.mb[0][2]; ++z)
                for (int y = 0; y < M.mb[0][1]; ++y)
                    for (int x = 0; x < M.mb[0][0]; ++x)
                        if (!M.m[0][((size_t)z * M.mb[0][1] + y) * M.mb[0][0] + x]) {
                            const int ax = x > bx ? x - bx : bx - x, ay = y > by ? y - by : by - y, az = z > bz ? z - bz : bz - z;
                            const int m = ax > ay ? (ax > az ? ax : az) : (ay > az ? ay : az);
                            if (m < dd) dd = m;
                        }
            dd -= 1;
            const int lox = ((bx - dd) << msh) > 0 ? ((bx - dd) << msh) : 0, loy = ((by - dd) << msh) > 0 ? ((by - dd) << msh) : 0,
                      loz = ((bz - dd) << msh) > 0 ? ((bz - dd) << msh) : 0;
            const int hix = ((bx + dd + 1) << msh) < nx ? ((bx + dd + 1) << msh) : nx,
                      hiy = ((by + dd + 1) << msh) < ny ? ((by + dd + 1) << msh) : ny,
                      hiz = ((bz + dd + 1) << msh) < nz ? ((bz + dd + 1) << msh) : nz;
            nf += mcrt::box_jump(ix, iy, iz, tmx, tmy, tmz, t, p[0], p[1], p[2], ivx, ivy, ivz, u[0], u[1], u[2], stx,
                                 sty, stz, lox, loy, loz, hix, hiy, hiz);
            ++nj;
            continue;
        }
        if (use_jumps == 1 && !d && M.empty(0, ix, iy, iz)) {
            int sh = msh;
            if (M.empty(2, ix, iy, iz)) sh = msh + 4;
            else if (M.empty(1, ix, iy, iz)) sh = msh + 2;
            const int lox = (ix >> sh) << sh, loy = (iy >> sh) << sh, loz = (iz >> sh) << sh;
            const int e = 1 << sh;
            const int hix = lox + e < nx ? lox + e : nx, hiy = loy + e < ny ? loy + e : ny, hiz = loz + e < nz ? loz + e : nz;
            nf += mcrt::box_jump(ix, iy, iz, tmx, tmy, tmz, t, p[0], p[1], p[2], ivx, ivy, ivz, u[0], u[1], u[2], stx,
                                 sty, stz, lox, loy, loz, hix, hiy, hiz);
            ++nj;
            continue;
        }
        const bool selx = (tmx <= tmy) && (tmx <= tmz);
        const bool sely = !selx && (tmy <= tmz);
        const double tn = selx ? tmx : (sely ? tmy : tmz);
        if (d) {
            if (cnt < max_n) { cells[cnt] = ((int64_t)iz * ny + iy) * nx + ix; ds_out[cnt] = tn - t; }
            ++cnt;
        }
        t = tn;
        ++nf;
        if (selx) { ix += stx; tmx = mcrt::face_t(ix, stx, p[0], ivx); }
        else if (sely) { iy += sty; tmy = mcrt::face_t(iy, sty, p[1], ivy); }
        else { iz += stz; tmz = mcrt::face_t(iz, stz, p[2], ivz); }
    }
    *faces = nf; *t_exit = t; *jumps = nj;
    return cnt;
}

}  // extern "C"
