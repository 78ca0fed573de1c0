// dda.h -- geometry of the cell walk (S4 of DESIGN.md): face parameters and the O(1) jump over a box of
// empty cells.  Shared by the CUDA kernels (mcrt.cu) and by the host-side unit test driver
// (dda_host.cpp, built by tests/test_dda_host.py); holds no physics.
//
// The paper only says that a packet "enters a neighboring cell according to its direction of travel"
// (PAPER.md:51).  Reading Q8: Amanatides-Woo traversal in which the parameter of a
// face is always computed from the face coordinate itself,
//        t_a(f) = (f - p_a) * (1/u_a),
// measured from the flight origin p in cell units.  The walk is then exactly the 3-way merge of the three
// per-axis face sequences ordered by (t, axis) -- x before y before z on equal t -- and a run of faces
// inside a box of vacuum cells can be crossed in one step with the identical result: box_jump() below.
//
// All arithmetic here must round like the oracle's: compile without FMA contraction
// (nvcc -fmad=false, g++ -ffp-contract=off).
#pragma once

#include <math.h>

#if defined(__CUDACC__)
#define MCRT_HD __host__ __device__ __forceinline__
#else
#define MCRT_HD inline
#endif

namespace mcrt {

// int -> double without the conversion pipe: 2^52 + 2^31 + (i xor 2^31) is exact, subtracting the bias
// leaves i.  Valid for every 32-bit i.
MCRT_HD double int_to_double(int i)
{
#if defined(__CUDA_ARCH__)
    return __hiloint2double(0x43300000, (int)((unsigned)i ^ 0x80000000u)) - 4503601774854144.0;
#else
    return (double)i;
#endif
}

// parameter of the face through which a packet leaves cell coordinate c along one axis
// (st = sign of the direction component, p = flight origin, inv = 1/u); +inf when st == 0
MCRT_HD double face_t(int c, int st, double p, double inv)
{
    if (st == 0) return (double)INFINITY;
    return (int_to_double(c + (st > 0 ? 1 : 0)) - p) * inv;
}

// Number of faces f_k = c + [st>0] + st*k, k = 0..K-1, along one axis whose (t, axis) sorts before the
// exit event (Te, exit axis): t_k < Te, or t_k == Te when this axis comes before the exit axis.
// t_k is non-decreasing in k (the subtraction and the product round monotonically), so the count is found
// from an estimate of the exit position and corrected with the exact predicate.
MCRT_HD int faces_before(int c, int st, double p, double inv, double u, int K, double Te, bool before_on_tie)
{
    if (st == 0 || K <= 0) return 0;
    // estimate: coordinate reached at Te, clamped so that the conversion to int is always defined
    double pos = p + Te * u;
    const double lo = (double)(c - K - 2), hi = (double)(c + K + 2);
    pos = fmin(fmax(pos, lo), hi);            // fmax/fmin drop a NaN estimate
    int k = (st > 0) ? ((int)floor(pos) - c) : (c - (int)ceil(pos) + 1);
    k = k < 0 ? 0 : (k > K ? K : k);
    const int f0 = c + (st > 0 ? 1 : 0);
    for (;;) {                                // faces the estimate missed
        if (k >= K) break;
        const double tk = (int_to_double(f0 + st * k) - p) * inv;
        if (!(tk < Te || (before_on_tie && tk == Te))) break;
        ++k;
    }
    for (;;) {                                // faces the estimate counted too many
        if (k <= 0) break;
        const double tk = (int_to_double(f0 + st * (k - 1)) - p) * inv;
        if (tk < Te || (before_on_tie && tk == Te)) break;
        --k;
    }
    return k;
}

// Cross, in one step, every face the cell-by-cell walk would cross until it leaves the box of cells
// [lox,hix) x [loy,hiy) x [loz,hiz) that contains the current cell (ix,iy,iz).  The caller guarantees that
// the walk would neither interact nor tally inside the box (all its cells are vacuum).
// On return: (ix,iy,iz) = first cell outside the box (possibly outside the grid), t = parameter of the
// exit face, tm* = parameters of the faces through which the new cell will be left.  Returns the number
// of faces crossed, the exit face included.
MCRT_HD unsigned box_jump(int &ix, int &iy, int &iz, double &tmx, double &tmy, double &tmz, double &t,
                          double px, double py, double pz, double ivx, double ivy, double ivz,
                          double ux, double uy, double uz, int stx, int sty, int stz,
                          int lox, int loy, int loz, int hix, int hiy, int hiz)
{
    const double Tx = face_t(stx > 0 ? hix - 1 : lox, stx, px, ivx);
    const double Ty = face_t(sty > 0 ? hiy - 1 : loy, sty, py, ivy);
    const double Tz = face_t(stz > 0 ? hiz - 1 : loz, stz, pz, ivz);
    const bool ex = (Tx <= Ty) && (Tx <= Tz);   // same rule as the cell walk: ties x < y < z
    const bool ey = !ex && (Ty <= Tz);
    const bool ez = !ex && !ey;
    const double Te = ex ? Tx : (ey ? Ty : Tz);
    // faces crossed on the exit axis, its box face included
    const int ce = ex ? ix : (ey ? iy : iz), ste = ex ? stx : (ey ? sty : stz);
    const int loe = ex ? lox : (ey ? loy : loz), hie = ex ? hix : (ey ? hiy : hiz);
    const int ne = (ste > 0) ? (hie - ce) : (ce - loe + 1);
    // the two other axes, in axis order: a1 = (x unless x exits, then y), a2 = (z unless z exits, then y).
    // A face of a1 / a2 that ties with the exit face comes first when its axis comes first.
    const int c1 = ex ? iy : ix, st1 = ex ? sty : stx, lo1 = ex ? loy : lox, hi1 = ex ? hiy : hix;
    const double p1 = ex ? py : px, iv1 = ex ? ivy : ivx, u1 = ex ? uy : ux;
    const int c2 = ez ? iy : iz, st2 = ez ? sty : stz, lo2 = ez ? loy : loz, hi2 = ez ? hiy : hiz;
    const double p2 = ez ? py : pz, iv2 = ez ? ivy : ivz, u2 = ez ? uy : uz;
    const int n1 = faces_before(c1, st1, p1, iv1, u1, (st1 > 0) ? (hi1 - 1 - c1) : (c1 - lo1), Te, !ex);
    const int n2 = faces_before(c2, st2, p2, iv2, u2, (st2 > 0) ? (hi2 - 1 - c2) : (c2 - lo2), Te, ez);
    ix += stx * (ex ? ne : n1);
    iy += sty * (ey ? ne : (ex ? n1 : n2));
    iz += stz * (ez ? ne : n2);
    tmx = face_t(ix, stx, px, ivx);
    tmy = face_t(iy, sty, py, ivy);
    tmz = face_t(iz, stz, pz, ivz);
    t = Te;
    return (unsigned)(ne + n1 + n2);
}

}  // namespace mcrt
