// mcrt.cu -- B200-native (sm_100a) photon-packet transport: C-ABI host layer + CUDA kernels.
//
// Implements include/mcrt.h.  Citations are lines of the paper text of Heymann &
// Siebenmorgen, arxiv 1203.2941.  Design notes, data layout and rooflines: DESIGN.md.
//
// Compile with -fmad=false: the fp64 trajectory arithmetic is written so that every product and sum is
// rounded separately (the parity contract with the CPU oracle).
//
// There is NO CPU fallback in this file: every step of the path (S0-S12 of DESIGN.md) runs in the
// kernels below; host code only builds the small lookup tables once and marshals arguments.
#include <cuda_runtime.h>
#include <math.h>
#include <math_constants.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <atomic>
#include <string>
#include <vector>

#include "mcrt.h"
#include "dda.h"

#define MCRT_VERSION_STRING "mcrt-b200 0.1 (sm_100a)"

// ------------------------------------------------------------------------------------------------
// constants
// ------------------------------------------------------------------------------------------------
namespace {

constexpr double kPlanckH = 6.62607015e-27;   // erg s
constexpr double kBoltzK = 1.380649e-16;      // erg K^-1
constexpr double kLightC = 2.99792458e10;     // cm s^-1
constexpr double kFourPi = 12.566370614359172953850573533118;

constexpr unsigned kFull = 0xffffffffu;
constexpr int kHot = 511;            // most hot cells around the source (see cw_hot)

enum : int { ST_IDLE = 0, ST_JUMP = 1, ST_INTERACT = 2, ST_FLY = 3, ST_DONE = 4, ST_STOP = 5, ST_SUB = 6 };
enum : int { EV_EMIT = 0, EV_SCATTER = 1, EV_ABSORB = 2, EV_ESCAPE = 3 };

// device counters (unsigned long long each)
enum : int { CNT_PACKETS = 0, CNT_CROSS, CNT_DUSTY, CNT_SCA, CNT_ABS, CNT_DIRECT, CNT_OVERFLOW, CNT_NEXT, CNT_CARRY, CNT_SCAEV, CNT_N };

thread_local std::string g_create_error;

}  // namespace

// A packet carried over an epoch boundary (NEXT-1; PAPER.md:128-130 restated deterministically, reading Q23): after
// carry_K interactions within one epoch a packet stops behind the carry_K-th (new direction and frequency drawn)
// and continues in the next epoch from this state, with its own random stream, at that epoch's temperatures.
struct CarryRec {
    unsigned long long pid, hash;
    double px, py, pz, ux, uy, uz;
    uint32_t w0, j, d, ncross, nsca, nabs;
};

// ------------------------------------------------------------------------------------------------
// context
// ------------------------------------------------------------------------------------------------
struct mcrt_ctx {
    int device = 0;
    cudaStream_t stream = 0;
    std::string err;
    // grid
    int nx = 0, ny = 0, nz = 0, ns = 0;
    int nbx = 0, nby = 0, nbz = 0;   // bricks per axis
    size_t nc = 0, ncp = 0;          // cells, cells of the padded storage (guard shell included)
    int px = 0, pxy = 0;             // row and plane pitch of the padded storage
    unsigned long long n_dusty = 0;  // cells with rho > 0
    uint32_t *d_hot_idx = nullptr;   // [kHot + 1] storage indices of the hot cells
    int n_hot = 0, hot_max = 31;
    uint32_t hot_shift = 24, hot_mask = 31, tidx_mask = 0xffffu;
    std::vector<uint32_t> hot_idx;   // [n_hot + 1]
    std::vector<uint32_t> hot_cand;  // storage indices of the dusty cells around the source, nearest first (<= hot_max)
    size_t l2_bytes = 126u << 20;
    double h = 0.0;
    // workspace (bump allocator)
    char *ws = nullptr;
    size_t ws_bytes = 0, ws_used = 0;
    bool ws_owned_by_caller = false;
    std::vector<void *> owned;       // cudaMalloc'ed blocks when no workspace was given
    // device arrays
    unsigned long long *cellw = nullptr;  // [ncp] packed cell words (see "Packed cell word")
    uint32_t *vmask = nullptr;            // vacuum mask: one bit per brick
    uint4 *vbox = nullptr;                // [bricks] a large box of empty bricks around every empty brick
    int *vsat = nullptr;                  // scratch: summed-area table of dusty bricks
    int msh = 2, mwords = 0;              // log2 brick edge; 32-bit words of the mask
    long long *lfx = nullptr;             // [ncp] Lucy fixed-point tally
    unsigned long long *kabs_cnt = nullptr, *kprev = nullptr;  // [ncp]
    void *scratch = nullptr;              // [nc*8 bytes]
    unsigned long long *counters = nullptr;  // [CNT_N]
    unsigned long long *sed = nullptr, *sed_direct = nullptr;  // [ndir*nf]
    double *d_kext_h = nullptr, *d_kabs_fx = nullptr, *d_albedo = nullptr, *d_g = nullptr;  // [ns*nf]
    double *d_srccdf = nullptr, *d_dnu = nullptr, *d_J = nullptr, *d_Tg = nullptr, *d_cdfB = nullptr, *d_cdfdB = nullptr;
    double *d_mu = nullptr;
    mcrt_digest *dig = nullptr;
    uint64_t dig_cap = 0, dig_n = 0;
    // host tables
    int nf = 0, nT = 0, ndir = 1, ndir_alloc = 0;
    std::vector<double> nu, dnu, kabs, ksca, g, Tg, kext_h, kabs_h, albedo, J, cdfB, cdfdB, srccdf, mu_edges;
    std::vector<unsigned short> perm;     // Eytzinger position -> ascending position of a CDF row
    unsigned short *d_perm = nullptr;
    int nfs = 0;                          // row stride of the device CDF tables
    double L = 0.0, pos[3] = {0, 0, 0};
    bool have_tables = false, have_source = false, mu_dirty = true;
    double *sed_stage = nullptr;          // [ndir*nf] staging of the SED for host reads
    // run state: fx / xi are the fixed-point scale and packet energy of the STORED tallies
    uint64_t last_n = 0;
    int fx = 40;
    double xi = 0.0;
    uint64_t epochs = 0, launches = 0;
    uint64_t dig_base = 0;                // packet id of digest slot 0
    int8_t *d_sca_slot = nullptr;                  // scattering-event store (cudaMalloc)
    mcrt_scatter_event *sca_ev = nullptr;
    uint64_t sca_cap = 0;
    std::vector<int> sca_bins;
    double *img_buf = nullptr; size_t img_cap = 0; // ray tracer: images and per-species opacity staging (cudaMalloc)
    CarryRec *carry_buf[2] = {nullptr, nullptr};   // carried packets: read by this epoch / written for the next (cudaMalloc)
    size_t carry_cap[2] = {0, 0};
    int carry_cur = 0;
    // dust mixtures (mcrt_dust_mixtures; NEXT-3): the species byte of a cell names a mixture of one or two materials
    bool mix = false;
    std::vector<int> mx_ncomp, mx_mat;             // [ns], [ns][2]
    std::vector<double> mx_frac, mx_S0, mx_A0, kabs1_h;   // [ns][2]; [ns*nf] event thresholds, f_1 kabs_1 h
    int *d_mx_ncomp = nullptr, *d_mx_mat = nullptr;       // device copies and the second component's per-cell arrays (cudaMalloc)
    double *d_mx_frac = nullptr, *d_mx_thr = nullptr, *d_kabs1_fx = nullptr;   // d_mx_thr: [ns*nf] {S0, A0}
    long long *lfx1 = nullptr;
    unsigned long long *kcnt1 = nullptr, *kprev1 = nullptr;
    uint16_t *tidx1 = nullptr;
    // sub-cubes (mcrt_subgrid; NEXT-3): refined cubes carry a marker word with their block number; their sub-cubes' arrays (cudaMalloc)
    int subR = 0, sub_shift = 0;
    size_t n_sub = 0, n_subcells = 0;
    unsigned long long *sub_cellw = nullptr, *sub_kcnt = nullptr, *sub_kprev = nullptr;
    long long *sub_lfx = nullptr;
    // thresholded Lucy estimator (mcrt_run_opts.lucy_hybrid; Sect. 3.1)
    bool hybrid = false;                           // the stored tallies were made with it
    double *d_kmax_diag = nullptr;                 // [ns] sqrt(3) h max_nu (kabs + ksca) (cudaMalloc)
    // run in progress (mcrt_run_begin .. mcrt_run_end)
    struct Run {
        bool active = false;
        mcrt_run_opts o;
        uint64_t n = 0, seed = 0, done = 0, Bnom = 0, Bprev = 0, Bmax = 0;
        int e = 0, sweep = 0, blocks = 0, threads = 0, prev_fx = 40;
        size_t smem = 0;
        double cellfac = 0.0, prev_cellfac = 0.0, growth = 2.0;
        bool finished = false;            // every step has been issued
        uint32_t carry_K = 0;             // interaction budget of the current epoch (0 = no carry-over)
        uint64_t n_carry = 0;             // packets carried into the next epoch
        int xtra = 0;                     // which rarely used features are in use (template argument XTRA of k_transport)
        bool hot = false;                 // hot cells tallied per CTA
    } run;
    bool need_exchange = false;           // partitioned run: a step's tallies are still per-part
    bool exchange_open = false, exchange_full = false;
    bool globalised = false;              // the stored tallies are sums over the parts of a partitioned run
    int occ_blocks = 0;
    // optional per-kernel timing: events e[3i], e[3i+1], e[3i+2] bracket update and transport of launch pair i
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    double transport_ms = 0.0, update_ms = 0.0;
};

namespace {

int fail(mcrt_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}

#define CUDA_TRY(c, expr)                                                                          \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess)                                                                    \
            return fail((c), MCRT_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e__));     \
    } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// record the next timing event on the context's stream (no-op unless timing is on)
void mark(mcrt_ctx *c, bool on)
{
    if (!on) return;
    if (c->ev_used == c->ev_pool.size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return;
        c->ev_pool.push_back(e);
    }
    cudaEventRecord(c->ev_pool[c->ev_used++], c->stream);
}

// fold the recorded (start, after-update, after-transport) triples into the running sums
void fold_timing(mcrt_ctx *c)
{
    for (size_t i = 0; i + 2 < c->ev_used; i += 3) {
        float a = 0.f, b = 0.f;
        if (cudaEventElapsedTime(&a, c->ev_pool[i], c->ev_pool[i + 1]) == cudaSuccess) c->update_ms += a;
        if (cudaEventElapsedTime(&b, c->ev_pool[i + 1], c->ev_pool[i + 2]) == cudaSuccess) c->transport_ms += b;
    }
    c->ev_used = 0;
}

int ws_alloc(mcrt_ctx *c, void **out, size_t bytes)
{
    bytes = align_up(bytes ? bytes : 1, 256);
    if (c->ws) {
        if (c->ws_used + bytes > c->ws_bytes)
            return fail(c, MCRT_ENOMEM, "workspace too small: need " + std::to_string(c->ws_used + bytes) +
                                            " bytes, have " + std::to_string(c->ws_bytes));
        *out = c->ws + c->ws_used;
        c->ws_used += bytes;
        return MCRT_OK;
    }
    void *p = nullptr;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) return fail(c, MCRT_ENOMEM, std::string("cudaMalloc: ") + cudaGetErrorString(e));
    c->owned.push_back(p);
    *out = p;
    return MCRT_OK;
}

// ------------------------------------------------------------------------------------------------
// device helpers
// ------------------------------------------------------------------------------------------------

// S1  Philox-4x32-10 (Salmon et al. 2011): counter-based, so a packet's stream depends only on
// (seed, packet id, draw index, pass) and never on scheduling.  Replaces the per-thread Mersenne
// Twister streams of PAPER.md:126.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}

// one block -> two uniforms strictly inside (0,1): zeta = (2*u52+1) * 2^-53
#ifndef MCRT_PHILOX_INLINE
#define MCRT_PHILOX_INLINE 1        // 0: one out-of-line copy of the generator (smaller code; measured 2 % slower on
#endif                              //    torus256 than the inlined copies: the calls cost more than the cache misses)
#if MCRT_PHILOX_INLINE
__device__ __forceinline__
#else
__device__ __noinline__
#endif
void draw2(uint32_t seed_lo, uint32_t seed_hi, unsigned long long pid, uint32_t d,
                                      uint32_t pass, double &z0, double &z1)
{
    uint32_t w0, w1, w2, w3;
    philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), d, pass, seed_lo, seed_hi, w0, w1, w2, w3);
    const unsigned long long a = (((unsigned long long)w0 << 32) | w1) >> 12;
    const unsigned long long b = (((unsigned long long)w2 << 32) | w3) >> 12;
    z0 = __ull2double_rn(2ull * a + 1ull) * 0x1.0p-53;
    z1 = __ull2double_rn(2ull * b + 1ull) * 0x1.0p-53;
}

// Elementary functions of the trajectory (reading Q28).  tau = -ln zeta and the azimuth
// 2 pi zeta are evaluated by explicit fp64 algorithms -- only + - * / on doubles, each rounded
// separately (this file is compiled with -fmad=false), fixed order -- so that the result does not depend on a
// math library's last ulp.  Coefficients are the correctly rounded doubles of 1/(2k+1) and of 1/n!.
//
// ln z, z a positive normal double: z = m 2^e, m in (sqrt(1/2), sqrt(2)]; ln m = 2 atanh(s), s = (m-1)/(m+1),
// Taylor series up to s^25 (Horner in s^2); ln 2 = hi + lo with e * hi exact.
__device__ __forceinline__ double traj_log(double z)
{
    int hi = __double2hiint(z);
    const int lo = __double2loint(z);
    int e = ((hi >> 20) & 0x7ff) - 1023;
    double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, lo);
    if (m > 0x1.6a09e667f3bcdp+0) { m = m * 0.5; e += 1; }
    const double f = m - 1.0;
    const double s = f / (2.0 + f);
    const double w = s * s;
    double p = 0x1.47ae147ae147bp-5;       // 1/25
    p = p * w + 0x1.642c8590b2164p-5;      // 1/23
    p = p * w + 0x1.8618618618618p-5;      // 1/21
    p = p * w + 0x1.af286bca1af28p-5;      // 1/19
    p = p * w + 0x1.e1e1e1e1e1e1ep-5;      // 1/17
    p = p * w + 0x1.1111111111111p-4;      // 1/15
    p = p * w + 0x1.3b13b13b13b14p-4;      // 1/13
    p = p * w + 0x1.745d1745d1746p-4;      // 1/11
    p = p * w + 0x1.c71c71c71c71cp-4;      // 1/9
    p = p * w + 0x1.2492492492492p-3;      // 1/7
    p = p * w + 0x1.999999999999ap-3;      // 1/5
    p = p * w + 0x1.5555555555555p-2;      // 1/3
    const double t = s * (w * p);
    const double lm = 2.0 * s + 2.0 * t;
    const double ed = (double)e;
    return (ed * 0x1.62e42fee00000p-1 + lm) + ed * 0x1.a39ef35793c76p-33;
}

// sin and cos of 2 pi z, z in [0, 1): q = round(4 z) quarter turns, r = 4 z - q in [-1/2, 1/2] (both exact),
// x = r pi/2, Taylor series to x^19 / x^18 (Horner in x^2), then the quadrant q mod 4.
__device__ __forceinline__ void traj_sincos_turns(double z, double &sn, double &cs)
{
    const double a = 4.0 * z;
    const double qd = floor(a + 0.5);
    const double r = a - qd;
    const double x = r * 0x1.921fb54442d18p+0;
    const double w = x * x;
    double p = -0x1.2f49b46814157p-57;     // -1/19!
    p = p * w + 0x1.952c77030ad4ap-49;     // +1/17!
    p = p * w - 0x1.ae7f3e733b81fp-41;     // -1/15!
    p = p * w + 0x1.6124613a86d09p-33;     // +1/13!
    p = p * w - 0x1.ae64567f544e4p-26;     // -1/11!
    p = p * w + 0x1.71de3a556c734p-19;     // +1/9!
    p = p * w - 0x1.a01a01a01a01ap-13;     // -1/7!
    p = p * w + 0x1.1111111111111p-7;      // +1/5!
    p = p * w - 0x1.5555555555555p-3;      // -1/3!
    const double s = x + x * (w * p);
    double c = -0x1.6827863b97d97p-53;     // -1/18!
    c = c * w + 0x1.ae7f3e733b81fp-45;     // +1/16!
    c = c * w - 0x1.93974a8c07c9dp-37;     // -1/14!
    c = c * w + 0x1.1eed8eff8d898p-29;     // +1/12!
    c = c * w - 0x1.27e4fb7789f5cp-22;     // -1/10!
    c = c * w + 0x1.a01a01a01a01ap-16;     // +1/8!
    c = c * w - 0x1.6c16c16c16c17p-10;     // -1/6!
    c = c * w + 0x1.5555555555555p-5;      // +1/4!
    c = c * w - 0.5;                       // -1/2!
    const double co = 1.0 + w * c;
    const int q = (int)qd & 3;
    sn = (q == 0) ? s : (q == 1) ? co : (q == 2) ? -s : -co;
    cs = (q == 0) ? co : (q == 1) ? -s : (q == 2) ? -co : s;
}

// smallest j with cdf[j] >= z (Eq. 5 / Eq. 10: "the shortest frequency nu' for which ...")
__device__ __forceinline__ int lower_bound_cdf(const double *cdf, int n, double z)
{
    int lo = 0, hi = n - 1;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (cdf[mid] >= z) hi = mid; else lo = mid + 1;
    }
    return lo;
}

// -DMCRT_CHECK=1: a debug build in which every index the transport kernel computes is checked before it is used
// (compute-sanitizer is not available on the pool this was developed on); a violation prints its site and traps.
#ifndef MCRT_CHECK
#define MCRT_CHECK 0
#endif
#if MCRT_CHECK
#define MCRT_CHK(cond, what)                                                                                              \
    do {                                                                                                                  \
        if (!(cond)) {                                                                                                    \
            printf("MCRT_CHECK failed: %s (line %d, block %d thread %d)\n", what, __LINE__, (int)blockIdx.x, (int)threadIdx.x); \
            __trap();                                                                                                     \
        }                                                                                                                 \
    } while (0)
#else
#define MCRT_CHK(cond, what) do { } while (0)
#endif
// L1 policy of the walk's cell-word loads and of the event phase's table loads (CDF rows, empty boxes).  Measured
// (profiles/r02_experiments.md, section 6): cell words kept longest +0.3-0.8 %; tables kept out of L1 -3 %.
#ifndef MCRT_TABLE_POLICY
#define MCRT_TABLE_POLICY ""
#endif
// Two walk-loop variants that lost (profiles/r02_experiments.md, section 6), kept selectable:
//   MCRT_ROT4         four steps per iteration with the two words in flight rotating through four registers and
//                     unpredicated loads (no copy and no wait for the loads at the end of an iteration): -6.5 %
//   MCRT_STOP_RELOAD  a stopped packet's cell word is loaded again instead of being stored at the stop: -5 %
#ifndef MCRT_ROT4
#define MCRT_ROT4 0
#endif
#ifndef MCRT_STOP_RELOAD
#define MCRT_STOP_RELOAD 0
#endif
#ifndef MCRT_CW_POLICY
#define MCRT_CW_POLICY ".L1::evict_last"
#endif
__device__ __forceinline__ double ldg_table(const double *p)
{
    double v;
    asm volatile("ld.global.nc" MCRT_TABLE_POLICY ".f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ uint4 ldg_table(const uint4 *p)
{
    uint4 v;
    asm volatile("ld.global.nc" MCRT_TABLE_POLICY ".v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
// The same lower bound on a row stored in Eytzinger (breadth-first) order, 1-based, the row 128-byte aligned: the
// first four levels of the search (entries 1..15) share one cache line, so a search costs about four round trips to
// L2 instead of seven or eight.  perm[k] = position of entry k in ascending order.
__device__ __forceinline__ int lower_bound_eytzinger(const double *__restrict__ row, const unsigned short *__restrict__ perm, int n, double z)
{
    int k = 1;
    while (k <= n) k = 2 * k + ((ldg_table(row + k) < z) ? 1 : 0);
    k >>= __ffs(~k);
    return (int)perm[k];
}

__device__ __forceinline__ void hash_mix(unsigned long long &h, unsigned long long w)
{
    h = (h ^ w) * 0x100000001B3ull;
}

__device__ __forceinline__ unsigned long long event_word(int type, int j, unsigned long long cell)
{
    return (unsigned long long)type | ((unsigned long long)j << 8) | (cell << 24);
}

// ------------------------------------------------------------------------------------------------
// Packed cell word (8 bytes, one per cell, brick-major order):
//   the fp64 bit pattern of the cell's fp32 density -- exact, its low 29 mantissa bits are always zero --
//   with the dust species in bits 0-7 and the frozen-epoch temperature index in bits 8-23.
// One 8-byte load per crossing serves S4, S5, S6 and S9, and the density needs no fp32->fp64 conversion.
// ------------------------------------------------------------------------------------------------
constexpr unsigned long long kRhoMask = 0xFFFFFFFFE0000000ull;
// kCS = stride of the cell-word array and of the Lucy-tally array in 8-byte words.  1: two separate arrays (default).
// 2: one 16-byte record per cell, so that the walk's load of a cell and its tally add two steps later touch the same
// 32-byte sector.  Measured (profiles/r02_experiments.md): disk256 +17 %, but torus256 -15 %, torus512 -18 %,
// shell128 -61 % -- a RED into the sector a cell word lives in keeps evicting it from L1 and serialises with its
// reads in L2, which costs far more where cells are revisited than the saved DRAM sector gains where they are not.
#ifndef MCRT_PITCH_ALIGN
#define MCRT_PITCH_ALIGN 1            // the row pitch of the padded storage is a multiple of this many cells
#endif
#ifndef MCRT_CELL_STRIDE
#define MCRT_CELL_STRIDE 1
#endif
constexpr int kCS = MCRT_CELL_STRIDE;
// The walk keeps kDepthReg cell words in flight per lane, in registers (its geometry runs that many cells ahead of the
// physics).  Round 1 kept them in a cp.async ring in shared memory: its groups complete in order, so any depth is
// one wait on one scoreboard, whereas ptxas gives the two register loads the same scoreboard.  Both were measured
// this round at depths 2-4 on all five workloads (profiles/r02_experiments.md, commits b3e3664..0e8480c carry the
// ring as `walk_words = 2`): the ring was never faster, not even on the grids that wait for DRAM -- it costs 9
// shared-memory wavefronts per step on the SM's busiest unit -- and was removed.
#ifndef MCRT_DEPTH
#define MCRT_DEPTH 2
#endif
constexpr int kDepthReg = MCRT_DEPTH;
constexpr int kGuard = kDepthReg + 1;  // guard cells around the grid (see "Storage order")

__device__ __forceinline__ double cw_rho(unsigned long long cw) { return __longlong_as_double((long long)(cw & kRhoMask)); }
__device__ __forceinline__ int cw_species(unsigned long long cw) { return (int)((unsigned)cw & 0xffu); }
__device__ __forceinline__ int cw_tidx(unsigned long long cw, uint32_t tmask) { return (int)(((unsigned)cw >> 8) & tmask); }
// Hot cells (north_star item 5; "local copies"): every packet starts in the few cells around the source,
// so their tallies are same-address atomics from every SM at once, which one L2 slice serialises.  The dusty cells
// nearest to the source are numbered 1, 2, ... in the bits of their cell word between the temperature index and the
// density (mcrt_source: bits 20-28, 511 cells, when the temperature grid has at most 4096 points; else bits 24-28,
// 31 cells) and tallied in a copy per CTA in shared memory, flushed with one atomic per CTA at the end of a launch.
// Integer adds: the result is the same.
__device__ __forceinline__ uint32_t cw_hot(unsigned long long cw, uint32_t shift, uint32_t mask) { return ((uint32_t)cw >> shift) & mask; }
__device__ __forceinline__ bool cw_vacuum(unsigned long long cw) { return (unsigned)(cw >> 32) == 0u; }  // rho == +0
// a cell that holds dust: 0 < rho < +inf (the cells of an empty brick carry the marker density +inf)
__device__ __forceinline__ bool cw_dusty(unsigned long long cw) { return (unsigned)(cw >> 32) - 1u < 0x7FEFFFFFu; }

// The grid is stored brick-major: bricks of E^3 cells, E = 1 << bsh (4 for grids up to 256^3, 8 up to 512^3),
// so that a packet's next cell is usually in the same 128-byte line or at least in the same brick.
//
// Vacuum masks: three bit arrays, level l = 0,1,2, one bit per aligned box of (E << 2l)^3 cells, set when
// every cell of the box (clipped to the grid) has rho == 0.  A level-0 box IS a brick, so the brick number
// of a cell indexes both its mask bit and its storage.  Level 0 lives in shared memory: cells of an empty
// brick are never loaded.
struct TransportParams {
    const unsigned long long *__restrict__ cellw;
    long long *__restrict__ lfx;
    unsigned long long *__restrict__ kcnt;
    const double *__restrict__ kext_h, *__restrict__ kabs_fx, *__restrict__ albedo, *__restrict__ g;
    const double *__restrict__ srccdf, *__restrict__ cdf, *__restrict__ mu_edges;
    const uint32_t *__restrict__ vmask;   // one bit per brick: every cell of the brick has rho == 0
    const uint4 *__restrict__ vbox;       // per empty brick: box of empty bricks {lox|loy<<16, loz|hix<<16, hiy|hiz<<16, -}
    unsigned long long *__restrict__ sed, *__restrict__ sed_direct, *__restrict__ counters;
    mcrt_digest *__restrict__ dig;
    int nx, ny, nz, ns, nf, nT, ndir;
    int nfs;            // stride of a re-emission CDF row (Eytzinger order, padded to 16 doubles)
    const unsigned short *__restrict__ perm;   // [nf + 1] Eytzinger position -> ascending position
    int nbx, nby;       // bricks per axis
    uint32_t ncp;       // padded cell count
    const uint32_t *__restrict__ hot_idx;   // [kHot + 1] storage index of hot cell number i (entry 0 unused)
    uint32_t hot_shift, hot_mask, tidx_mask;   // fields of the cell word's low half: species 0-7 | T index | hot number | rho 29-31
    int n_hot;
    int lpx, lpxy;      // row and plane pitch of the padded storage
    double inv_lpx, inv_lpxy;
    int bsh;            // log2 of the brick edge
    int mwords;         // 32-bit words of the mask
    double px, py, pz;  // source position, cell units
    unsigned long long pid0, count, dig_base, dig_n;
    const CarryRec *__restrict__ carry_in;     // packets carried over from the previous epoch: taken before new ids
    CarryRec *__restrict__ carry_out;          // packets whose budget runs out in this launch (counters[CNT_CARRY] of them)
    uint32_t n_carry_in, carry_K;              // carry_K = 0: no budget
    uint32_t source_strata;                    // > 0: stratified source frequencies (Eq. 1)
    int live_bw;                               // 1: the temperature index follows every absorption, not the epoch
    const double *__restrict__ J;              // [ns][nT] left side of Eq. 4 (live_bw)
    double cellfac;                            // xi / (4 pi V) (live_bw)
    const int8_t *__restrict__ sca_slot;       // [nf] slot of a stored frequency bin (-1: not stored), or NULL
    mcrt_scatter_event *__restrict__ sca_ev;   // the event list and its capacity; counters[CNT_SCAEV] counts
    unsigned long long sca_cap;
    // dust mixtures (NEXT-3; readings Q34-Q36): NULL lfx1 = the species byte names a material
    long long *__restrict__ lfx1;              // Lucy tally, absorption count and temperature index of the second component
    unsigned long long *__restrict__ kcnt1;
    const uint16_t *__restrict__ tidx1;
    const double *__restrict__ kabs1_fx;       // [ns][nf] f_1 kabs_1 h 2^FX (0 for a one-component mixture)
    const double2 *__restrict__ mx_thr;        // [ns][nf] {S0, A0}: thresholds of the event uniform
    const int *__restrict__ mx_mat;            // [ns][2] material of each component
    // thresholded Lucy estimator (Sect. 3.1, readings Q37 / Q38): NULL = the linear tally in every cell
    // sub-cubes (NEXT-3, reading Q40): subR = 0 none.  A refined cube's cell word is a marker with kSubFlag and its block
    // number << kSubShift; sub-cube (gx, gy, gz) of block b is cell b R^3 + (gz R + gy) R + gx of the sub arrays
    int subR, sub_shift;
    const unsigned long long *__restrict__ sub_cellw;
    long long *__restrict__ sub_lfx;
    unsigned long long *__restrict__ sub_kcnt;
    unsigned long long sub_n;                  // number of sub-cubes
    unsigned long long nc_grid;                // cells of the grid: a sub-cube's number in digests is nc_grid + its index
    int redraw;                                // 1: a new optical depth is drawn on entering every cell (as printed)
    const double *__restrict__ kmax_diag;      // [ns] sqrt(3) h max_nu (kabs + ksca): a cell is tallied if rho * this < 10^-2
    double two_fx, inv_two_fx;                 // 2^FX, 2^-FX
    uint32_t seed_lo, seed_hi, pass;
};

// full brick-major index of cell (ix, iy, iz)
__device__ __forceinline__ uint32_t brick_of(int ix, int iy, int iz, int nbx, int nby, int bsh)
{
    return (uint32_t)((iz >> bsh) * nby + (iy >> bsh)) * (uint32_t)nbx + (uint32_t)(ix >> bsh);
}
// storage index of cell (ix, iy, iz) (see "Storage order")
__device__ __forceinline__ uint32_t lin_index(int ix, int iy, int iz, int px, int pxy)
{
    return (uint32_t)((iz + kGuard) * pxy + (iy + kGuard) * px + (ix + kGuard));
}
// ... and back, for a cell inside the grid: packed coordinates (quotients by a reciprocal, corrected exactly)
__device__ __forceinline__ uint32_t index_to_packed(uint32_t idx, uint32_t px, uint32_t pxy, double inv_px, double inv_pxy)
{
    uint32_t z = __double2uint_rz(__uint2double_rn(idx) * inv_pxy);
    int r = (int)(idx - z * pxy);
    if (r < 0) { --z; r += (int)pxy; }
    if (r >= (int)pxy) { ++z; r -= (int)pxy; }
    uint32_t y = __double2uint_rz(__uint2double_rn((uint32_t)r) * inv_px);
    int x = r - (int)(y * px);
    if (x < 0) { --y; x += (int)px; }
    if (x >= (int)px) { ++y; x -= (int)px; }
    return (uint32_t)(x - kGuard) | ((y - (uint32_t)kGuard) << 11) | ((z - (uint32_t)kGuard) << 22);
}
__device__ __forceinline__ bool brick_empty(const uint32_t *__restrict__ m0, uint32_t brick) { return (m0[brick >> 5] >> (brick & 31u)) & 1u; }


// S5 Lucy path-length tally: L[c] += rint(x), x = kabs h rho ds 2^FX >= 0 (Eq. 9, linear form;
// PAPER.md:142 integer atomics).  rint by the 1.5 * 2^52 trick: round to nearest even, exact below 2^51, and
// x < 37 * 2^40 always, because a packet never spends more than its tau = -ln zeta <= 36.8 in one cell.
__device__ __forceinline__ unsigned long long lucy_round(double x)
{
    // round to nearest even by adding 1.5 * 2^52: the integer sits in the mantissa, the bias in the high word only
    const double y = x + 6755399441055744.0;
    return ((unsigned long long)(uint32_t)(__double2hiint(y) - 0x43380000) << 32) | (uint32_t)__double2loint(y);
}
__device__ __forceinline__ void lucy_add_raw(long long *__restrict__ lfx, uint32_t cidx, unsigned long long q)
{
    asm volatile("red.global.add.u64 [%0], %1;" ::"l"(lfx + (size_t)kCS * cidx), "l"(q) : "memory");
}
// Eq. 9, per traversal of a cell below the threshold of Sect. 3.1: (1 - e^-tau) 2^FX from the linear
// tally value x = tau 2^FX; 1 - e^-tau is DEFINED as its series to tau^5 in this order (reading Q38; tau < 10^-2)
constexpr double kThinTau = 1e-2;
__device__ __forceinline__ double eq9_fx(double x, double two_fx, double inv_two_fx)
{
    const double tau = x * inv_two_fx;
    return (tau * (1.0 - tau * (0.5 - tau * (1.0 / 6.0 - tau * (1.0 / 24.0 - tau * (1.0 / 120.0)))))) * two_fx;
}
__device__ __forceinline__ void lucy_add(long long *__restrict__ lfx, uint32_t cidx, double x)
{
    const unsigned long long q = lucy_round(x);
    // (explicitly global: a pointer that went through shared memory has lost its address space)
    asm volatile("red.global.add.u64 [%0], %1;" ::"l"(lfx + (size_t)kCS * cidx), "l"(q) : "memory");
}

// Warp aggregation of these adds (__match_any_sync + __reduce_add_sync per group) was measured slower everywhere:
// 2.5-5x in the cell walk, and in the event phase the groups are almost always single lanes, whose reductions
// then run one after the other (7 % of the kernel's stall samples).  Plain RED atomics: L2 does the sums.

// ------------------------------------------------------------------------------------------------
// S0-S10  the transport kernel: persistent CTAs; every warp owns a POOL of kSlots packets in shared memory.
//
// A packet is either FLYING (walking cell by cell towards its next interaction), JUMPING (inside a run of empty
// bricks) or waiting for an EVENT (emission of the slot's next packet, an interaction, the escape tally).  The
// three kinds of work share no code, so a warp never mixes them: it alternates between
//   S phase: the 32 lanes check flying packets out of the pool into registers and step them cell by cell (S4/S5);
//            lanes whose packet stopped are refilled from the pool MCRT_SWAP_MIN at a time, and the rest is parked
//            again when the pool has nothing left for MCRT_S_LEAVE idle lanes;
//   J phase: up to 32 jumping packets cross their runs of empty bricks box by box (mcrt::box_jump, dda.h);
//   E phase: entered when fewer than 32 packets can fly; the lanes take up to 32 waiting packets and each
//            performs that packet's event (S1-S3, S6-S10; S0 refill: one atomic per warp for the new packet ids).
// With 64 packets per warp both phases run with (nearly) all lanes active whatever the mix of optical
// depths -- the scheduling-independent replacement of the paper's pause/resume balancer.
// Results never depend on which lane or warp carries a packet: all random numbers are Philox blocks keyed
// by (seed, packet id, draw index, pass) and all tallies are integer atomics.
// ------------------------------------------------------------------------------------------------
#ifndef MCRT_SLOTS
#define MCRT_SLOTS 64
#endif
constexpr int kSlots = MCRT_SLOTS;  // packets per warp (<= 128: the slot sets are one or two 64-bit masks)
#ifndef MCRT_SLOT_IV
#define MCRT_SLOT_IV 0              // 1: the slot also holds 1/u per axis (computed once per direction, not per refill)
#endif
constexpr int kSlotF64 = 11 + 3 * MCRT_SLOT_IV;   // 8-byte fields per slot (+1, the digest hash, in the recording kernel)
constexpr int kSlotU32 = 6;         // 4-byte fields per slot
__host__ __device__ constexpr int pool_bytes_per_warp(bool record) { return kSlots * ((kSlotF64 + (record ? 1 : 0)) * 8 + kSlotU32 * 4); }
#ifndef MCRT_MAX_THREADS
#define MCRT_MAX_THREADS 640        // 20 warps per SM at <= 96 registers per thread (512 threads / 128 registers: 1 % slower)
#endif
#ifndef MCRT_SWAP_MIN
#define MCRT_SWAP_MIN 8             // S phase: stopped packets are parked / replaced this many lanes at a time
#endif
#ifndef MCRT_PIN
#define MCRT_PIN 3                  // how many of the walk loop's kernel parameters are pinned in registers (1..3)
#endif
#ifndef MCRT_S_ENTER
#define MCRT_S_ENTER 32             // an S phase starts when the pool holds this many flying packets
#endif
#ifndef MCRT_S_LEAVE
#define MCRT_S_LEAVE 8              // ... and ends when this many lanes are idle and nothing is left to refill them
#endif
#ifndef MCRT_J_MIN
#define MCRT_J_MIN 10               // a J phase ends when fewer lanes than this still jump
#endif
#ifndef MCRT_SMEM_MASK
#define MCRT_SMEM_MASK 0            // 1: every CTA keeps a copy of the empty-brick mask in shared memory; 0: read through L1
#endif

#if MCRT_SLOT_IV
enum : int { F_PX = 0, F_PY, F_PZ, F_UX, F_UY, F_UZ, F_T, F_TAU, F_ZTYPE, F_CW, F_PID, F_IVX, F_IVY, F_IVZ, F_HASH };
#else
enum : int { F_PX = 0, F_PY, F_PZ, F_UX, F_UY, F_UZ, F_T, F_TAU, F_ZTYPE, F_CW, F_PID, F_HASH };
#endif
// MCRT_PACK_STOP = 1: what a stopping packet stores in the walk sits in adjacent words of its slot -- (t, tau) as one
// 16-byte pair, (crossings, cell) as one 8-byte pair -- so that a stop is three shared-memory stores instead of five
#ifndef MCRT_J_ONELOAD
#define MCRT_J_ONELOAD 1            // 1: the jump loop reads the landing brick's box entry (its fourth word says "empty") instead of
#endif                              //    the mask bit and then the box: one dependent load per jump instead of two
#ifndef MCRT_L2_HINT
#define MCRT_L2_HINT 0              // 1: the walk's cell-word loads carry an L2 evict_last policy; 2: and its tally REDs evict_first
#endif
#ifndef MCRT_PF
#define MCRT_PF 0                   // > 0: the walk prefetches into L2 a guessed cell this many iterations (of kDepth cells) ahead
#endif
#ifndef MCRT_VAC_SPECIES
#define MCRT_VAC_SPECIES 0          // 1: vacuum cells inside dusty bricks take the species byte of the nearest dusty cell (k_vac_species)
#endif
#ifndef MCRT_VAC_KEEP
#define MCRT_VAC_KEEP 0             // 1: a vacuum cell does not reload the walk's cached opacities (its species byte is irrelevant)
#endif
#ifndef MCRT_PACK_STOP
#define MCRT_PACK_STOP 0
#endif
#if MCRT_PACK_STOP
enum : int { U_DK = 0, U_NCROSS, U_W0, U_NSCA, U_NABS, U_W1 };   // DK = draw counter | kind << 30
#else
enum : int { U_DK = 0, U_NCROSS, U_NSCA, U_NABS, U_W0, U_W1 };   // DK = draw counter | kind << 30
#endif
enum : uint32_t { K_EMIT = 0u, K_INTERACT = 1u, K_ESCAPED = 2u };
// cell coordinates packed in 32 bits: x, y < 2048, z < 1024
__device__ __forceinline__ uint32_t pack_xyz(int x, int y, int z) { return (uint32_t)x | ((uint32_t)y << 11) | ((uint32_t)z << 22); }
__device__ __forceinline__ int unpack_x(uint32_t w) { return (int)(w & 0x7ffu); }
__device__ __forceinline__ int unpack_y(uint32_t w) { return (int)((w >> 11) & 0x7ffu); }
__device__ __forceinline__ int unpack_z(uint32_t w) { return (int)(w >> 22); }
// Marker words: density +inf.  The cell words of an empty brick carry it ("a run of empty bricks starts here"), and
// so does the word stored behind the grid that stands for every cell outside it (with kOutFlag in the temperature
// field).  The walk needs no test of its own for them: rho = +inf makes the optical depth of the cell infinite.
constexpr unsigned long long kJumpWord = 0x7FF0000000000000ull;
constexpr uint32_t kMarkHi = 0x7FF00000u, kOutFlag = 0x100u;
constexpr unsigned long long kOutWord = kJumpWord | kOutFlag;
// ... and so does the word of a cube that is divided into sub-cubes (mcrt_subgrid): kSubFlag and its block number
constexpr uint32_t kSubFlag = 0x200u;
constexpr int kSubShift = 10;
// state of a packet inside a divided cube, kept in the upper half of slot word U_W1: sub-cube coordinates, "valid"
constexpr uint32_t kSubOk = 1u << 25;
__device__ __forceinline__ uint32_t sub_pack(int gx, int gy, int gz) { return kSubOk | ((uint32_t)gx << 16) | ((uint32_t)gy << 19) | ((uint32_t)gz << 22); }
// Storage order of the per-cell arrays (cell words, Lucy tally, absorption counts): linear, x fastest, with a shell
// of kGuard cells around the grid that hold the "outside the grid" marker word:
//     index(ix, iy, iz) = ((iz + kGuard) * PY + (iy + kGuard)) * PX + (ix + kGuard),  PX = nx + 2 kGuard, PY = ny + 2 kGuard.
// A step of the walk along one axis is then one constant added to the index (+-1, +-PX, +-PX*PY), a cell outside
// the grid needs no test (its word says so), and the geometry of the walk may run up to kGuard cells beyond the grid.

// position of the n-th set bit (n = 0, 1, ...) of a 64-bit mask; n < popc(m)
__device__ __forceinline__ int nth_set64(unsigned long long m, int n)
{
    const uint32_t lo = (uint32_t)m, hi = (uint32_t)(m >> 32);
    const int clo = __popc(lo);
    const bool up = n >= clo;
    const uint32_t w = up ? hi : lo;
    n = up ? n - clo : n;
    int pos = 0;
#pragma unroll
    for (int sft = 16; sft; sft >>= 1) {
        const int c = __popc((w >> pos) & ((1u << sft) - 1u));
        if (n >= c) { n -= c; pos += sft; }
    }
    return pos + (up ? 32 : 0);
}

// warp-wide OR of one 64-bit word per lane
__device__ __forceinline__ unsigned long long warp_or64(unsigned long long v)
{
    const uint32_t lo = __reduce_or_sync(kFull, (uint32_t)v), hi = __reduce_or_sync(kFull, (uint32_t)(v >> 32));
    return ((unsigned long long)hi << 32) | lo;
}

// A set of pool slots, warp-uniform (every lane holds the same value): one or two 64-bit masks.
constexpr int kSetWords = (kSlots + 63) / 64;
struct SlotSet {
    unsigned long long w[kSetWords];
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int i = 0; i < kSetWords; ++i) w[i] = 0ull;
    }
    __device__ __forceinline__ void fill() {   // slots 0 .. kSlots-1
#pragma unroll
        for (int i = 0; i < kSetWords; ++i) {
            const int n = kSlots - 64 * i;
            w[i] = n >= 64 ? ~0ull : ((1ull << (n & 63)) - 1ull);
        }
    }
    __device__ __forceinline__ int count() const {
        int c = 0;
#pragma unroll
        for (int i = 0; i < kSetWords; ++i) c += __popcll(w[i]);
        return c;
    }
    __device__ __forceinline__ bool empty() const {
        unsigned long long a = 0ull;
#pragma unroll
        for (int i = 0; i < kSetWords; ++i) a |= w[i];
        return a == 0ull;
    }
    // slot number of the n-th member (n = 0, 1, ...; n < count())
    __device__ __forceinline__ int nth(int n) const {
        if (kSetWords == 1) return nth_set64(w[0], n);
        const int c0 = __popcll(w[0]);
        return n < c0 ? nth_set64(w[0], n) : 64 + nth_set64(w[kSetWords - 1], n - c0);
    }
    // every lane with on == true contributes its slot: add them to / remove them from the set (warp-wide)
    __device__ __forceinline__ void add(bool on, int slot) {
#pragma unroll
        for (int i = 0; i < kSetWords; ++i) w[i] |= warp_or64((on && (slot >> 6) == i) ? (1ull << (slot & 63)) : 0ull);
    }
    __device__ __forceinline__ void remove(bool on, int slot) {
#pragma unroll
        for (int i = 0; i < kSetWords; ++i) w[i] &= ~warp_or64((on && (slot >> 6) == i) ? (1ull << (slot & 63)) : 0ull);
    }
};

__device__ __forceinline__ int t_index(const double *J, int nT, double x);

// 64-bit add into a per-CTA hot-cell tally kept as two 32-bit limbs (native shared atomics; a 64-bit one is a CAS
// loop): the carry out of the low limb goes into the high limb's add.  The limbs are put together at the flush.
__device__ __forceinline__ void hot_add(unsigned int *hot, uint32_t id, unsigned long long q)
{
    unsigned int *t = hot + 3u * id;
    const unsigned int ql = (unsigned int)q, old = atomicAdd(t, ql);
    const unsigned int carry = (old + ql < old) ? 1u : 0u;
    const unsigned int qh = (unsigned int)(q >> 32) + carry;
    if (qh) atomicAdd(t + 1, qh);
}
// shared-memory words of the hot-cell tallies (entry 0 unused), a whole number of 16-byte units
__host__ __device__ constexpr int hot_smem_words(int n_hot) { return (3 * (n_hot + 1) + 3) & ~3; }
constexpr int kPermSmem = 1024;

// XTRA: 0 = none of the rarely used features; 1 = those that live outside the walk loop (carry-over, event store, stratified
// source, live B&W, sub-cubes); 2 = those of 1 and the ones inside it (mixtures, thresholded estimator); 3 = those of 2
// and the per-cell redraw of the optical depth (a Philox block and a logarithm in every step)
template <bool RECORD, bool HOT, int XTRA>
__global__ void __launch_bounds__(MCRT_MAX_THREADS, 1) k_transport(const TransportParams P)
{
    constexpr int kDepth = kDepthReg;
    extern __shared__ double2 smem_d2[];
    // Per-CTA tallies of the hot cells, at the START of the dynamic shared memory (compile-time addresses): three
    // words per cell -- the two limbs of the 64-bit Lucy tally and the absorption count.
    unsigned int *s_hot = reinterpret_cast<unsigned int *>(smem_d2);
    const int hot_words = HOT ? hot_smem_words(P.n_hot) : 0;
    if (HOT) for (int i = threadIdx.x; i < hot_words; i += blockDim.x) s_hot[i] = 0u;
    const int nsf = P.ns * P.nf;
    const int nwarps = blockDim.x >> 5;
    constexpr int kPoolF64 = pool_bytes_per_warp(RECORD) / 8;
    constexpr int kNF64 = kSlotF64 + (RECORD ? 1 : 0);
    double *s_pool = reinterpret_cast<double *>(s_hot + hot_words);      // [nwarps][pool_bytes_per_warp]
    double2 *s_kk = reinterpret_cast<double2 *>(s_pool + (size_t)nwarps * kPoolF64);
    double2 *s_ag = s_kk + nsf;              // {albedo, g};  s_kk = {kext_h, kabs_fx}: one LDS.128 per crossing
    double *s_src = reinterpret_cast<double *>(s_ag + nsf);
    double *s_mu = s_src + P.nf;
    unsigned long long *s_cnt = reinterpret_cast<unsigned long long *>(s_mu + P.ndir + 1);
    unsigned int *s_hist = reinterpret_cast<unsigned int *>(s_cnt + 8 * nwarps);
    const int nhist = 2 * P.ndir * P.nf;
    uint32_t *s_m0x = s_hist + nhist;        // level-0 vacuum mask (one bit per brick)
    const int mw_smem = MCRT_SMEM_MASK ? P.mwords : 0;
    // Eytzinger permutation of the frequency grid (grids of kPermSmem points and more read P.perm instead)
    unsigned short *s_perm = reinterpret_cast<unsigned short *>(s_m0x + ((mw_smem + 1) & ~1));
    if (P.nf < kPermSmem) for (int i = threadIdx.x; i <= P.nf; i += blockDim.x) s_perm[i] = P.perm[i];
    const uint32_t *s_m0 = MCRT_SMEM_MASK ? s_m0x : P.vmask;

    for (int i = threadIdx.x; i < nsf; i += blockDim.x) {
        s_kk[i] = make_double2(P.kext_h[i], P.kabs_fx[i]);
        s_ag[i] = make_double2(P.albedo[i], P.g[i]);
    }
    for (int i = threadIdx.x; i < P.nf; i += blockDim.x) s_src[i] = P.srccdf[i];
    for (int i = threadIdx.x; i <= P.ndir; i += blockDim.x) s_mu[i] = P.mu_edges[i];
    for (int i = threadIdx.x; i < nhist; i += blockDim.x) s_hist[i] = 0u;
    for (int i = threadIdx.x; i < mw_smem; i += blockDim.x) s_m0x[i] = P.vmask[i];
    for (int i = threadIdx.x; i < 8 * nwarps; i += blockDim.x) s_cnt[i] = 0ull;   // eight counters per warp
    // Kernel parameters the walk loop uses, parked in shared memory: the S phase reads them into registers through
    // a volatile pointer, so that they stay there (left to itself the compiler reloads a dozen of them from the
    // constant bank in every iteration of the loop and waits for them)
    __shared__ unsigned long long s_parp[2];
    __shared__ uint32_t s_pari[8];
    if (threadIdx.x == 0) {
        s_parp[0] = reinterpret_cast<unsigned long long>(P.cellw);
        s_parp[1] = reinterpret_cast<unsigned long long>(P.lfx);
        s_pari[0] = P.ncp; s_pari[1] = (uint32_t)P.nbx; s_pari[2] = (uint32_t)P.nby; s_pari[3] = (uint32_t)P.nx;
        s_pari[4] = (uint32_t)P.ny; s_pari[5] = (uint32_t)P.lpx; s_pari[6] = (uint32_t)P.lpxy; s_pari[7] = (uint32_t)P.nf;
    }
    __syncthreads();

    const int lane = (int)(threadIdx.x & 31u);
    const int nf = P.nf, bsh = P.bsh, nbx = P.nbx, nby = P.nby, lpx = P.lpx, lpxy = P.lpxy;
    double *wf = s_pool + (size_t)(threadIdx.x >> 5) * kPoolF64;                  // this warp's pool, f64 fields
    uint32_t *wu = reinterpret_cast<uint32_t *>(wf + kNF64 * kSlots);             // its u32 fields
#if MCRT_PACK_STOP
    static_assert(F_TAU == F_T + 1 && U_W0 == U_NCROSS + 1, "the pairs stored at a stop are neighbouring fields");
#define SF(f, s) wf[((f) == F_T || (f) == F_TAU) ? F_T * kSlots + 2 * (s) + ((f) - F_T) : (f) * kSlots + (s)]
#define SU(f, s) wu[((f) == U_NCROSS || (f) == U_W0) ? U_NCROSS * kSlots + 2 * (s) + ((f) - U_NCROSS) : (f) * kSlots + (s)]
#else
#define SF(f, s) wf[(f) * kSlots + (s)]
#define SU(f, s) wu[(f) * kSlots + (s)]
#endif

    // every slot starts as "emit the next packet"
    for (int s = lane; s < kSlots; s += 32) SU(U_DK, s) = K_EMIT << 30;
    __syncwarp();
    // warp-uniform slot sets: parked flying packets / packets inside a run of empty bricks / packets waiting for an event
    SlotSet mFly, mJ, mEv;
    SlotSet mSub;                                  // packets inside a cube divided into sub-cubes (XTRA kernels only)
    mSub.clear();
    mFly.clear(); mJ.clear(); mEv.fill();
    bool exhausted = false;                        // the epoch counter has run out (warp-uniform)
    uint32_t ndusty_acc = 0u;                      // dusty crossings stepped by this lane

    for (;;) {
        const int nfly = mFly.count(), njmp = mJ.count(), nevt = mEv.count(), nsub = XTRA ? mSub.count() : 0;
        if (nfly >= MCRT_S_ENTER || (nfly > 0 && njmp == 0 && nevt == 0 && nsub == 0)) {
            // =========================================================== S phase: S4/S5 cell walk
            // Software pipeline.  The path of a flight does not depend on the cells' contents, so the geometry
            // (G: axis choice, next cell, exit parameter) runs ahead of the physics: in the step that handles cell n,
            // G enters cell n+2 and issues the load of its word into a register (two words are in flight per lane,
            // wA / wB, which alternate in the two steps of the loop body), so the latency of a cell word is covered
            // by two walk steps of every resident warp.  Between G and the physics sits one queue entry (exit
            // parameter and storage index of cell n+1).
            // Lanes whose packet reaches an event or an empty brick park it and take another flying packet
            // from the pool without leaving the loop; a new packet enters the pipeline behind one no-op cell
            // (zero length, vacuum), which the physics passes without effect.  The phase ends when the pool has
            // no flying packet left for MCRT_S_LEAVE idle lanes.
            int slot = 0, state = ST_IDLE;
            double px = 0.0, py = 0.0, pz = 0.0, ivx = 0.0, ivy = 0.0, ivz = 0.0, tmx = 0.0, tmy = 0.0, tmz = 0.0;
            double tau = 0.0;
            double tprev = 0.0, tnA = 0.0;                      // parameters at which cell n is entered and left
            double fdx = 0.0, fdy = 0.0, fdz = 0.0;             // coordinate of the face through which G's cell is left
            int shx = 0, shy = 0, shz = 0;                      // high word of the step per axis as a double (+1, -1 or 0)
            uint32_t gi = 0u, ciA = 0u;                         // storage index of G's cell and of cell n
            uint32_t dgx = 0u, dgy = 0u, dgz = 0u;              // the step per axis as an increment of the storage index
            uint32_t ncross = 0u;
            double2 kq = make_double2(0.0, 0.0);                // {kext_h, kabs_fx} of species kq_sp at the packet's frequency
            uint32_t kq_sp = 0u;
            const double2 *kq_row = s_kk;                       // s_kk + j
            const double *k1_row = P.kabs1_fx;                  // mixtures: the second component's kabs_fx at frequency j
            double kq1 = 0.0;
            double kmd = 0.0;                                   // thresholded estimator: kmax_diag of species kq_sp
            unsigned long long rd_pid = 0ull;                   // per-cell redraw: the packet's id and its draw index minus crossings
            uint32_t rd_base = 0u;
            // words of cells n .. n+kDepth-1, in registers
            unsigned long long cwr[kDepth];
            unsigned long long wstop = 0ull;             // cell word of the cell this lane's packet stopped in (MCRT_STOP_RELOAD)
#pragma unroll
            for (int i = 0; i < kDepth; ++i) cwr[i] = 0ull;
            double tq[kDepth - 1];                              // queue between G and the physics: exit parameter and storage
            uint32_t cq[kDepth - 1];                            // index of cells n+1 .. n+kDepth-2 (and of the cell G is in)
#pragma unroll
            for (int i = 0; i < kDepth - 1; ++i) { tq[i] = 0.0; cq[i] = 0u; }
            int nidle = 32;
            const volatile unsigned long long *vpp = s_parp;
            const volatile uint32_t *vpi = s_pari;
            const unsigned long long *const cellw_r = reinterpret_cast<const unsigned long long *>(vpp[0]);
            // L2 policies (MCRT_L2_HINT): cell words, which the walk waits for, stay in L2 longest; tally lines go first
            unsigned long long l2_keep = 0ull, l2_stream = 0ull;
            if (MCRT_L2_HINT) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(l2_keep));
            if (MCRT_L2_HINT == 2) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(l2_stream));
            long long *const lfx_r = reinterpret_cast<long long *>(vpp[1]);
            const uint32_t px_r = vpi[5], pxy_r = vpi[6];
            const uint32_t nf_r = vpi[7];

            for (;;) {
                // ---- account for packets that stopped, refill idle lanes (batched: MCRT_SWAP_MIN lanes at a time)
                {
                    if (state == ST_STOP) {
                        // stopped in the walk below, which stored the flight's state in the slot; what kind of stop is
                        // read off the cell word: a marker word (rho = +inf) is a cell outside the grid (bit 8) or the
                        // first cell of a run of empty bricks, anything else an interaction in that cell
#if MCRT_STOP_RELOAD
                        const unsigned long long scw = wstop;
                        SF(F_CW, slot) = __longlong_as_double((long long)scw);
#else
                        const unsigned long long scw = (unsigned long long)__double_as_longlong(SF(F_CW, slot));
#endif
                        const bool mk = (uint32_t)(scw >> 32) == kMarkHi;
                        state = mk ? (((uint32_t)scw & kOutFlag) ? ST_DONE : ST_JUMP) : ST_INTERACT;
                        if (XTRA && mk && ((uint32_t)scw & kSubFlag)) state = ST_SUB;   // a cube divided into sub-cubes
                        if (state == ST_DONE) SU(U_DK, slot) = (SU(U_DK, slot) & 0x3fffffffu) | (K_ESCAPED << 30);
                        else {
                            SU(U_W0, slot) = index_to_packed(SU(U_W0, slot), px_r, pxy_r, P.inv_lpx, P.inv_lpxy);   // the walk stored the index
                            if (state == ST_INTERACT) SU(U_DK, slot) = (SU(U_DK, slot) & 0x3fffffffu) | (K_INTERACT << 30);
                        }
                    }
                    mJ.add(state == ST_JUMP, slot);
                    if (XTRA) mSub.add(state == ST_SUB, slot);
                    mEv.add(state == ST_DONE || state == ST_INTERACT, slot);
                    if (state != ST_FLY) state = ST_IDLE;
                    const unsigned idle = __ballot_sync(kFull, state == ST_IDLE);
                    const int nfl = 32 - __popc(idle);
                    // nothing left to refill with and many lanes idle: let the other phases make flying packets
                    if (mFly.empty() && (nfl == 0 || (nfl <= 32 - MCRT_S_LEAVE && !(mJ.empty() && mEv.empty() && mSub.empty())))) {
                        // park mid-flight: cell n, entered at tprev.  A packet still behind its no-op cell has not
                        // started: its slot is as the refill found it
                        // (its crossing count is still below the slot's)
                        if (state == ST_FLY && (int)(ncross - SU(U_NCROSS, slot)) >= 0) {
                            const unsigned long long wn = cwr[0];
                            SU(U_NCROSS, slot) = ncross;
                            if (wn == kOutWord) {      // cell n lies outside the grid: the packet has escaped
                                SU(U_DK, slot) = (SU(U_DK, slot) & 0x3fffffffu) | (K_ESCAPED << 30);
                                state = ST_DONE;
                            } else {
                                SF(F_T, slot) = tprev; SF(F_TAU, slot) = tau;
                                SF(F_CW, slot) = __longlong_as_double((long long)wn);
                                SU(U_W0, slot) = index_to_packed(ciA, px_r, pxy_r, P.inv_lpx, P.inv_lpxy);
                            }
                        }
                        mFly.add(state == ST_FLY, slot);
                        mEv.add(state == ST_DONE, slot);
                        break;
                    }
                    const int k = __popc(idle & ((1u << lane) - 1u));
                    const bool take = state == ST_IDLE && k < mFly.count();
                    if (take) {
                        slot = mFly.nth(k);
                        px = SF(F_PX, slot); py = SF(F_PY, slot); pz = SF(F_PZ, slot);
                        {   // 1/u per axis (reading Q8); +inf for a zero direction component: that axis never moves
#if MCRT_SLOT_IV
                            ivx = SF(F_IVX, slot); ivy = SF(F_IVY, slot); ivz = SF(F_IVZ, slot);
#else
                            const double ux = SF(F_UX, slot), uy = SF(F_UY, slot), uz = SF(F_UZ, slot);
                            ivx = (ux != 0.0) ? 1.0 / ux : CUDART_INF;
                            ivy = (uy != 0.0) ? 1.0 / uy : CUDART_INF;
                            ivz = (uz != 0.0) ? 1.0 / uz : CUDART_INF;
#endif
                        }
                        const double t = SF(F_T, slot);
                        tau = SF(F_TAU, slot);
                        const uint32_t w0 = SU(U_W0, slot);
                        const int j = (int)(SU(U_W1, slot) & 0xffffu);   // (high half: interactions in this epoch)
                        ncross = SU(U_NCROSS, slot) - (uint32_t)(kDepth - 1);   // the no-op cells below count themselves
                        const int gx = unpack_x(w0), gy = unpack_y(w0), gz = unpack_z(w0);
                        // the stored 1/u is +inf for a zero direction component: that axis never moves
                        const int stx = isinf(ivx) ? 0 : (ivx > 0.0 ? 1 : -1);
                        const int sty = isinf(ivy) ? 0 : (ivy > 0.0 ? 1 : -1);
                        const int stz = isinf(ivz) ? 0 : (ivz > 0.0 ? 1 : -1);
                        tmx = mcrt::face_t(gx, stx, px, ivx);
                        tmy = mcrt::face_t(gy, sty, py, ivy);
                        tmz = mcrt::face_t(gz, stz, pz, ivz);
                        // an axis that never moves: f = +inf, so that (f - p) * (1/u) = inf * inf stays +inf
                        fdx = stx ? (double)(gx + ((stx + 1) >> 1)) : CUDART_INF; shx = __double2hiint((double)stx);
                        fdy = sty ? (double)(gy + ((sty + 1) >> 1)) : CUDART_INF; shy = __double2hiint((double)sty);
                        fdz = stz ? (double)(gz + ((stz + 1) >> 1)) : CUDART_INF; shz = __double2hiint((double)stz);
                        gi = lin_index(gx, gy, gz, (int)px_r, (int)pxy_r);
                        dgx = (uint32_t)stx; dgy = (uint32_t)(sty * (int)px_r); dgz = (uint32_t)(stz * (int)pxy_r);
                        // pipeline: kDepth - 1 no-op cells (zero length, vacuum word: nothing is tallied), then the packet's
                        // cell, in which G stands
#pragma unroll
                        for (int i = 0; i < kDepth - 1; ++i) cwr[i] = 0ull;
                        cwr[kDepth - 1] = (unsigned long long)__double_as_longlong(SF(F_CW, slot));
                        tprev = t; tnA = t; ciA = 0u;
#pragma unroll
                        for (int i = 0; i < kDepth - 2; ++i) { tq[i] = t; cq[i] = 0u; }
                        kq_row = s_kk + j;
                        kq_sp = 0u; kq = kq_row[0];
                        if (XTRA >= 2 && P.lfx1) { k1_row = P.kabs1_fx + j; kq1 = k1_row[0]; }
                        if (XTRA >= 2 && P.kmax_diag) kmd = P.kmax_diag[0];
                        if (XTRA >= 3 && P.redraw) {
                            rd_pid = (unsigned long long)__double_as_longlong(SF(F_PID, slot));
                            rd_base = SU(U_DK, slot) & 0x3fffffffu;
                        }
                        state = ST_FLY;
                    }
                    mFly.remove(take, slot);
                    nidle = __popc(__ballot_sync(kFull, state == ST_IDLE));
                }
                // ---- the walk: a tight inner loop (nothing but the step, so that it stays in the instruction cache)
                // until MCRT_SWAP_MIN more lanes have stopped.  kDepth cells per iteration, one per word in flight.
                //
                // No branch in a step: a divergent branch costs more here (branch resolution, reconvergence) than the
                // work it skips, so every lane runs the whole step.  A lane that holds no flying packet leaves no
                // trace: its G stands still and loads nothing, its physics works on whatever its registers
                // hold and tallies nothing.  A lane whose packet stops stores the flight's state in its slot at once
                // (predicated stores), so that nothing but `state` and `slot` has to survive until the next refill:
                // every other update of the step is unconditional.
                // Shared memory is touched only by the rare events of a step (stop, change of species): the step's
                // two global accesses (cell word, tally) already keep the SM's load/store data path busy.
                int nnot;
#define WALK_STEP(W, WN)                                                                                                         \
                {                                                                                                           \
                    const bool fly = state == ST_FLY;                                                                       \
                    const unsigned long long cw = W;                  /* the word of cell n (waits for its load) */        \
                    /* ---- G: the queue entry of cell n+1 (the cell G is in), then G advances to cell n+2 and loads its  */ \
                    /* word.  G stands still once its lane has stopped; until then it may run up to kGuard cells beyond  */ \
                    /* the grid (the storage has that many guard cells on every side).                                   */ \
                    const uint32_t ciN = gi;                                                                                \
                    const bool selx = (tmx <= tmy) && (tmx <= tmz);                                                         \
                    const bool sely = !selx && (tmy <= tmz);                                                                \
                    const bool selz = !selx && !sely;                                                                       \
                    const double tnN = selx ? tmx : (sely ? tmy : tmz);                                                     \
                    if (MCRT_ROT4) gi = fly ? gi + (selx ? dgx : (sely ? dgy : dgz)) : 0u;                                  \
                    else gi += fly ? (selx ? dgx : (sely ? dgy : dgz)) : 0u;                                                \
                    /* the load of cell n+kDepth replaces, in place, the word just read (lanes without a flying packet   */ \
                    /* keep theirs): tied to W, so that no move has to wait for the load                                  */ \
                    MCRT_CHK(!fly || gi < P.ncp, "walk: storage index of the prefetched cell");                             \
                    if (MCRT_ROT4) asm("ld.global.nc" MCRT_CW_POLICY ".u64 %0, [%1];" : "=l"(WN) : "l"(cellw_r + kCS * gi));     \
                    else                                                                                                    \
                    if (MCRT_L2_HINT)                                                                                       \
                    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p ld.global.nc" MCRT_CW_POLICY ".L2::cache_hint.u64 %0, [%1], %3;\n\t}" \
                                 : "+l"(W) : "l"(cellw_r + kCS * gi), "r"((uint32_t)fly), "l"(l2_keep));                   \
                    else                                                                                                    \
                    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p ld.global.nc" MCRT_CW_POLICY ".u64 %0, [%1];\n\t}" \
                                 : "+l"(W) : "l"(cellw_r + kCS * gi), "r"((uint32_t)fly));                                 \
                    /* parameter of the face through which the entered cell will be left (reading Q8): the face          */ \
                    /* coordinate f is kept as a double (integers are exact), t = (f - p) * (1/u).  The selected axis'   */ \
                    /* f moves by its step, the others by 0, and all three t are recomputed: the same value for an axis  */ \
                    /* that did not move, so nothing has to be selected afterwards                                       */ \
                    fdx += __hiloint2double(selx ? shx : 0, 0);                                                             \
                    fdy += __hiloint2double(sely ? shy : 0, 0);                                                             \
                    fdz += __hiloint2double(selz ? shz : 0, 0);                                                             \
                    tmx = (fdx - px) * ivx;                                                                                 \
                    tmy = (fdy - py) * ivy;                                                                                 \
                    tmz = (fdz - pz) * ivz;                                                                                 \
                    /* ---- physics of cell n.  One test for every kind of stop: a marker word (cell in an empty brick,  */ \
                    /* cell outside the grid) has rho = +inf, so dtau is +inf or (ds = 0) NaN                             */ \
                    const double ds = tnA - tprev;                                                                          \
                    const double rho_c = cw_rho(cw);                                                                        \
                    /* opacities of this cell's species at the packet's frequency; a vacuum cell needs none (rho = 0  */    \
                    /* makes every product 0 whatever kq holds), so it leaves the cached pair alone                    */    \
                    if (cw_species(cw) != kq_sp && (!MCRT_VAC_KEEP || __double2hiint(rho_c) != 0)) {                        \
                        kq_sp = cw_species(cw);                                                                             \
                        MCRT_CHK(!fly || kq_sp < (uint32_t)P.ns, "walk: species of the cell word");                         \
                        kq = kq_row[(fly || !MCRT_CHECK) ? kq_sp * nf_r : 0u];                                              \
                        if (XTRA >= 2 && P.lfx1) kq1 = k1_row[fly ? kq_sp * nf_r : 0u];   /* second component of a mixture */     \
                        if (XTRA >= 2 && P.kmax_diag) kmd = P.kmax_diag[fly ? kq_sp : 0u]; /* thresholded estimator */             \
                    }                                                                                                       \
                    if (XTRA >= 3 && P.redraw && fly) {   /* a new random number on entering the cell */             \
                        double zr0, zr1;                                                                                    \
                        draw2(P.seed_lo, P.seed_hi, rd_pid, (rd_base + ncross) & 0x3fffffffu, P.pass, zr0, zr1);            \
                        tau = -traj_log(zr0);                                                                               \
                    }                                                                                                       \
                    const double dtau = kq.x * rho_c * ds;            /* tau_i = (kabs+ksca) h rho ds (Eq. 2) */ \
                    const bool stop = !(dtau <= tau);                 /* interaction inside this cell: equality leaves (Q5) */ \
                    if (fly && stop) {                                                                                      \
                        state = ST_STOP;                                                                                    \
                        if (MCRT_PACK_STOP) {                                                                               \
                            *reinterpret_cast<uint2 *>(&SU(U_NCROSS, slot)) = make_uint2(ncross, ciA);                      \
                            *reinterpret_cast<double2 *>(&SF(F_T, slot)) = make_double2(tprev, tau);                        \
                        } else {                                                                                            \
                            SU(U_NCROSS, slot) = ncross; SU(U_W0, slot) = ciA;                                              \
                            SF(F_T, slot) = tprev; SF(F_TAU, slot) = tau;                                                   \
                        }                                                                                                   \
                        if (!MCRT_STOP_RELOAD) SF(F_CW, slot) = __longlong_as_double((long long)cw);                        \
                    }                                                                                                       \
                    /* the stopped packet's cell word is read again (rare; an L1 hit) instead of being kept: its register */ \
                    /* is then free for the load above, which otherwise needs a copy and a wait at the end of the loop  */ \
                    if (MCRT_STOP_RELOAD)                                                                                   \
                        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p ld.global.nc.u64 %0, [%1];\n\t}"      \
                                     : "+l"(wstop) : "l"(cellw_r + kCS * ciA), "r"((uint32_t)(fly && stop)));               \
                    /* S5: tally of a traversed dusty cell (a vacuum cell has nothing to add) */                           \
                    {                                                                                                       \
                        const bool hyb = XTRA >= 2 && P.kmax_diag;       /* Sect. 3.1: Eq. 9 in cells below the threshold only */ \
                        const double xq = kq.y * rho_c * ds;                                                                \
                        const unsigned long long q = lucy_round(hyb ? eq9_fx(xq, P.two_fx, P.inv_two_fx) : xq);             \
                        const bool go = fly && !stop;                                                                       \
                        const uint32_t dusty = (go && __double2hiint(rho_c) != 0) ? 1u : 0u;                                \
                        const uint32_t hid = HOT ? cw_hot(cw, P.hot_shift, P.hot_mask) : 0u;   /* tallied in the CTA's own copy */ \
                        const uint32_t cold = (dusty && hid == 0u && !(hyb && !(rho_c * kmd < kThinTau))) ? 1u : 0u;        \
                        MCRT_CHK(!dusty || ciA < P.ncp, "walk: storage index of the tallied cell");                         \
                        MCRT_CHK(hid <= (uint32_t)P.n_hot, "walk: hot-cell number");                                        \
                        MCRT_CHK(!(fly && stop) || (uint32_t)slot < (uint32_t)kSlots, "walk: slot of the stopped packet");   \
                        if (MCRT_L2_HINT == 2)                                                                              \
                        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p red.global.add.L2::cache_hint.u64 [%0], %1, %3;\n\t}" \
                                     ::"l"(lfx_r + kCS * ciA), "l"(q), "r"((HOT || XTRA >= 2) ? cold : dusty), "l"(l2_stream) : "memory"); \
                        else                                                                                                \
                        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p red.global.add.u64 [%0], %1;\n\t}"  \
                                     ::"l"(lfx_r + kCS * ciA), "l"(q), "r"((HOT || XTRA >= 2) ? cold : dusty) : "memory");       \
                        if (XTRA >= 2 && P.lfx1) {       /* the second component's tally (reading Q36) */                         \
                            const unsigned long long q1 = lucy_round(kq1 * rho_c * ds);                                     \
                            if (dusty && kq1 != 0.0) lucy_add_raw(P.lfx1, ciA, q1);                                         \
                        }                                                                                                   \
                        if (HOT && __any_sync(kFull, dusty && hid != 0u)) {                                                 \
                            if (dusty && hid != 0u) hot_add(s_hot, hid, q);                                    \
                        }                                                                                                   \
                        ndusty_acc += dusty;                                                                                \
                    }                                                                                                       \
                    tau -= dtau;                                                                                            \
                    ncross++;                                                                                               \
                    tprev = tnA;                                                                                            \
                    if (kDepth == 2) { tnA = tnN; ciA = ciN; }                                                              \
                    else {                                                                                                  \
                        tnA = tq[0]; ciA = cq[0];                                                                           \
                        _Pragma("unroll") for (int i = 0; i < kDepth - 3; ++i) { tq[i] = tq[i + 1]; cq[i] = cq[i + 1]; }    \
                        tq[kDepth - 3 >= 0 ? kDepth - 3 : 0] = tnN; cq[kDepth - 3 >= 0 ? kDepth - 3 : 0] = ciN;             \
                    }                                                                                                       \
                }
#if MCRT_ROT4
                static_assert(kDepth == 2, "the rotating walk loop is written for two words in flight");
                unsigned long long cw2, cw3;
                for (;;) {
                    WALK_STEP(cwr[0], cw2)
                    WALK_STEP(cwr[1], cw3)
                    nnot = __popc(__ballot_sync(kFull, state != ST_FLY));
                    if (nnot - nidle >= MCRT_SWAP_MIN || nnot == 32) { cwr[0] = cw2; cwr[1] = cw3; break; }
                    WALK_STEP(cw2, cwr[0])
                    WALK_STEP(cw3, cwr[1])
                    nnot = __popc(__ballot_sync(kFull, state != ST_FLY));
                    // (the empty statement gives this exit a block of its own: without it the copies that bring both
                    // exits' words into the same registers are placed in the loop, behind a wait for the loads)
                    if (nnot - nidle >= MCRT_SWAP_MIN || nnot == 32) { asm volatile(""); break; }
                }
#else
                do {
                    const uint32_t g_before = gi;
#pragma unroll
                    for (int i = 0; i < kDepth; ++i) WALK_STEP(cwr[i], cwr[i])
                    if (MCRT_PF) {
                        // A guess at where the ray will be MCRT_PF iterations on -- G's index moved on by the displacement
                        // of this iteration, as if the next steps took the same axes -- fetched into L2 ahead of time.
                        // Wrong guesses cost a sector of bandwidth and nothing else.
                        const uint32_t gp = gi + (uint32_t)MCRT_PF * (gi - g_before);
                        if (state == ST_FLY && gp < P.ncp)
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(cellw_r + kCS * gp));
                    }
                } while ((nnot = __popc(__ballot_sync(kFull, state != ST_FLY)), nnot - nidle < MCRT_SWAP_MIN && nnot != 32));
#endif
#undef WALK_STEP
            }
            __syncwarp();
        } else if (XTRA && nsub > 0 && nsub >= nevt && nsub >= njmp) {
            // =========================================================== R phase: cubes divided into sub-cubes (NEXT-3)
            // Each lane takes one packet that stands in a divided cube and walks its sub-cubes one by one -- the same
            // walk on the lattice of sub-cube faces f = c + k/R (reading Q40), not pipelined -- through any further
            // divided cubes, until it interacts (E phase), reaches an undivided cube (back to the pool) or escapes.
            const int nr = min(nsub, 32);
            const bool act = lane < nr;
            const int slot = act ? mSub.nth(lane) : 0;
            const int R = P.subR, R3 = R * R * R;
            const double Rd = (double)R;
            bool busy = act, escaped = false, hit = false;
            double px = 0.0, py = 0.0, pz = 0.0, ux = 0.0, uy = 0.0, uz = 0.0, ivx = 0.0, ivy = 0.0, ivz = 0.0;
            double t = 0.0, tau = 0.0, fx = 0.0, fy = 0.0, fz = 0.0;
            int ix = 0, iy = 0, iz = 0, gx = 0, gy = 0, gz = 0, stx = 0, sty = 0, stz = 0, j = 0;
            uint32_t ncross = 0u, blk = 0u, rbase = 0u;
            unsigned long long rpid = 0ull, fw = 0ull, pw = 0ull;
            bool g_ok = false, need_cube = true;
            if (act) {
                px = SF(F_PX, slot); py = SF(F_PY, slot); pz = SF(F_PZ, slot);
                ux = SF(F_UX, slot); uy = SF(F_UY, slot); uz = SF(F_UZ, slot);
                ivx = (ux != 0.0) ? 1.0 / ux : CUDART_INF;
                ivy = (uy != 0.0) ? 1.0 / uy : CUDART_INF;
                ivz = (uz != 0.0) ? 1.0 / uz : CUDART_INF;
                stx = (ux > 0.0) ? 1 : ((ux < 0.0) ? -1 : 0);
                sty = (uy > 0.0) ? 1 : ((uy < 0.0) ? -1 : 0);
                stz = (uz > 0.0) ? 1 : ((uz < 0.0) ? -1 : 0);
                t = SF(F_T, slot); tau = SF(F_TAU, slot);
                const uint32_t w0 = SU(U_W0, slot), w1 = SU(U_W1, slot);
                ix = unpack_x(w0); iy = unpack_y(w0); iz = unpack_z(w0);
                ncross = SU(U_NCROSS, slot);
                j = (int)(w1 & 0xffffu);
                g_ok = (w1 & kSubOk) != 0u;
                gx = (int)((w1 >> 16) & 7u); gy = (int)((w1 >> 19) & 7u); gz = (int)((w1 >> 22) & 7u);
                if (XTRA >= 3 && P.redraw) { rpid = (unsigned long long)__double_as_longlong(SF(F_PID, slot)); rbase = SU(U_DK, slot) & 0x3fffffffu; }
            }
            // (1/R is a power of two: the products below are the oracle's quotients (g + 1) / R, exactly.  The step is
            // written without branches on the axis: lanes of a warp take different axes, and a branch per axis made the
            // compiler's software division and the face arithmetic run lane by lane)
            const double invR = 1.0 / Rd;
            const int upx = stx > 0 ? 1 : 0, upy = sty > 0 ? 1 : 0, upz = stz > 0 ? 1 : 0;
            // The word of the NEXT position -- the next sub-cube's, or the next cube's when the step leaves this one -- is
            // loaded one step ahead (which position that is does not depend on what the sub-cubes hold): nw, valid if nw_ok.
            unsigned long long nw = 0ull;
            bool nw_ok = false;
            do {
                if (busy && need_cube) {
                    pw = nw_ok ? nw : __ldg(P.cellw + (size_t)kCS * lin_index(ix, iy, iz, lpx, lpxy));
                    nw_ok = false;
                    if (!((uint32_t)(pw >> 32) == kMarkHi && ((uint32_t)pw & kSubFlag))) { busy = false; g_ok = false; }
                    else {
                        blk = (uint32_t)pw >> kSubShift;
                        if (!g_ok) {   // entered from an undivided cube: the sub-cube that holds the entry point p + u t
                            int q;
                            q = (int)floor(((px + ux * t) - (double)ix) * Rd); gx = q < 0 ? 0 : (q > R - 1 ? R - 1 : q);
                            q = (int)floor(((py + uy * t) - (double)iy) * Rd); gy = q < 0 ? 0 : (q > R - 1 ? R - 1 : q);
                            q = (int)floor(((pz + uz * t) - (double)iz) * Rd); gz = q < 0 ? 0 : (q > R - 1 ? R - 1 : q);
                            g_ok = true;
                        }
                        need_cube = false;
                    }
                }
                if (busy) {
                    const uint32_t fidx = blk * (uint32_t)R3 + (uint32_t)((gz * R + gy) * R + gx);
                    MCRT_CHK(fidx < (uint32_t)P.sub_n, "sub-cube index");
                    fw = nw_ok ? nw : __ldg(P.sub_cellw + (size_t)kCS * fidx);
                    nw_ok = false;
                    // parameters of the faces through which sub-cube g is left: f = c + (g + [u > 0]) / R
                    fx = stx ? (((double)ix + (double)(gx + upx) * invR) - px) * ivx : CUDART_INF;
                    fy = sty ? (((double)iy + (double)(gy + upy) * invR) - py) * ivy : CUDART_INF;
                    fz = stz ? (((double)iz + (double)(gz + upz) * invR) - pz) * ivz : CUDART_INF;
                    const bool selx = (fx <= fy) && (fx <= fz), sely = !selx && (fy <= fz), selz = !selx && !sely;
                    const double tn = selx ? fx : (sely ? fy : fz);
                    const double ds = tn - t;
                    // where the packet goes if it does not stop here: the neighbouring sub-cube along the selected axis;
                    // through a face of the cube: the next cube, same row
                    int ngx = gx + (selx ? stx : 0), ngy = gy + (sely ? sty : 0), ngz = gz + (selz ? stz : 0);
                    const bool ox = (unsigned)ngx >= (unsigned)R, oy = (unsigned)ngy >= (unsigned)R, oz = (unsigned)ngz >= (unsigned)R;
                    ngx = ox ? (upx ? 0 : R - 1) : ngx; ngy = oy ? (upy ? 0 : R - 1) : ngy; ngz = oz ? (upz ? 0 : R - 1) : ngz;
                    const int nix = ix + (ox ? stx : 0), niy = iy + (oy ? sty : 0), niz = iz + (oz ? stz : 0);
                    const bool out = ox || oy || oz;
                    const bool esc = out && (((unsigned)nix >= (unsigned)P.nx) | ((unsigned)niy >= (unsigned)P.ny) | ((unsigned)niz >= (unsigned)P.nz));
                    if (!out) { nw = __ldg(P.sub_cellw + (size_t)kCS * (blk * (uint32_t)R3 + (uint32_t)((ngz * R + ngy) * R + ngx))); nw_ok = true; }
                    else if (!esc) { nw = __ldg(P.cellw + (size_t)kCS * lin_index(nix, niy, niz, lpx, lpxy)); nw_ok = true; }
                    // physics of this sub-cube
                    const double rho_c = cw_rho(fw);
                    const double2 kq = s_kk[cw_species(fw) * nf + j];
                    if (XTRA >= 3 && P.redraw) {
                        double zr0, zr1;
                        draw2(P.seed_lo, P.seed_hi, rpid, (rbase + ncross) & 0x3fffffffu, P.pass, zr0, zr1);
                        tau = -traj_log(zr0);
                    }
                    const double dtau = kq.x * rho_c * ds;
                    if (!(dtau <= tau)) { hit = true; busy = false; }
                    else {
                        tau -= dtau;
                        if (__double2hiint(rho_c) != 0) { lucy_add(P.sub_lfx, fidx, kq.y * rho_c * ds); ndusty_acc++; }
                        t = tn;
                        ncross++;
                        gx = ngx; gy = ngy; gz = ngz; ix = nix; iy = niy; iz = niz;
                        need_cube = out;
                        if (esc) { escaped = true; busy = false; }
                    }
                }
            } while (__popc(__ballot_sync(kFull, busy)) >= max(min(nr, MCRT_J_MIN), 1));
            bool to_jump = false;
            if (act) {
                SF(F_T, slot) = t; SF(F_TAU, slot) = tau;
                SU(U_NCROSS, slot) = ncross;
                const uint32_t w1 = SU(U_W1, slot) & 0xffffu;
                if (escaped) {
                    SU(U_DK, slot) = (SU(U_DK, slot) & 0x3fffffffu) | (K_ESCAPED << 30);
                    SU(U_W1, slot) = w1;
                } else {
                    SU(U_W0, slot) = pack_xyz(ix, iy, iz);
                    if (hit) {              // interaction inside sub-cube g: the E phase finds it by the flag in U_W1
                        SU(U_DK, slot) = (SU(U_DK, slot) & 0x3fffffffu) | (K_INTERACT << 30);
                        SF(F_CW, slot) = __longlong_as_double((long long)fw);
                        SU(U_W1, slot) = w1 | sub_pack(gx, gy, gz);
                    } else if (busy) {      // still inside: stays in the set
                        SU(U_W1, slot) = w1 | (need_cube ? (g_ok ? sub_pack(gx, gy, gz) : 0u) : sub_pack(gx, gy, gz));
                    } else {                // an undivided cube: back to the walk (or to the jumps, if its brick is empty)
                        SF(F_CW, slot) = __longlong_as_double((long long)pw);
                        SU(U_W1, slot) = w1;
                        to_jump = brick_empty(s_m0, brick_of(ix, iy, iz, nbx, nby, bsh));
                    }
                }
            }
            const bool mine = act && !busy;
            mSub.remove(mine, slot);
            mEv.add(mine && (escaped || hit), slot);
            mFly.add(mine && !escaped && !hit && !to_jump, slot);
            mJ.add(mine && !escaped && !hit && to_jump, slot);
            __syncwarp();
        } else if (njmp > 0 && njmp >= nevt) {
            // =========================================================== J phase: runs of empty bricks
            // Each lane takes one packet whose current cell lies in an empty brick and crosses, one box per
            // step, the largest aligned empty box around it (mcrt::box_jump, identical to the cell-by-cell
            // walk: same faces, same count, same exit parameter) until it reaches a brick that holds dust or
            // leaves the grid.  No global memory is touched on the way.
            const int nj = min(njmp, 32);
            const bool act = lane < nj;
            const int slot = act ? mJ.nth(lane) : 0;
            bool busy = act, escaped = false;
            double px = 0.0, py = 0.0, pz = 0.0, ivx = 0.0, ivy = 0.0, ivz = 0.0, ux = 0.0, uy = 0.0, uz = 0.0;
            double tmx = 0.0, tmy = 0.0, tmz = 0.0, t = 0.0;
            int ix = 0, iy = 0, iz = 0, stx = 0, sty = 0, stz = 0;
            uint32_t ncross = 0u;
            if (act) {
                px = SF(F_PX, slot); py = SF(F_PY, slot); pz = SF(F_PZ, slot);
                ux = SF(F_UX, slot); uy = SF(F_UY, slot); uz = SF(F_UZ, slot);
#if MCRT_SLOT_IV
                ivx = SF(F_IVX, slot); ivy = SF(F_IVY, slot); ivz = SF(F_IVZ, slot);
#else
                ivx = (ux != 0.0) ? 1.0 / ux : CUDART_INF;
                ivy = (uy != 0.0) ? 1.0 / uy : CUDART_INF;
                ivz = (uz != 0.0) ? 1.0 / uz : CUDART_INF;
#endif
                t = SF(F_T, slot);
                const uint32_t w0 = SU(U_W0, slot);
                ncross = SU(U_NCROSS, slot);
                ix = unpack_x(w0); iy = unpack_y(w0); iz = unpack_z(w0);
                stx = isinf(ivx) ? 0 : (ivx > 0.0 ? 1 : -1);
                sty = isinf(ivy) ? 0 : (ivy > 0.0 ? 1 : -1);
                stz = isinf(ivz) ? 0 : (ivz > 0.0 ? 1 : -1);
                tmx = mcrt::face_t(ix, stx, px, ivx);
                tmy = mcrt::face_t(iy, sty, py, ivy);
                tmz = mcrt::face_t(iz, stz, pz, ivz);
            }
            const int jmin = min(nj, MCRT_J_MIN);
            uint4 bb = make_uint4(0u, 0u, 0u, 0u);
            if (MCRT_J_ONELOAD && busy) bb = ldg_table(P.vbox + brick_of(ix, iy, iz, nbx, nby, bsh));
            do {
                if (busy) {
                    // the precomputed box of empty bricks around this brick, in cells, clipped to the grid
                    MCRT_CHK(ix >= 0 && iy >= 0 && iz >= 0 && ix < P.nx && iy < P.ny && iz < P.nz, "jump: cell coordinates");
                    if (!MCRT_J_ONELOAD) bb = ldg_table(P.vbox + brick_of(ix, iy, iz, nbx, nby, bsh));
                    const int lox = (int)(bb.x & 0xffffu) << bsh, loy = (int)(bb.x >> 16) << bsh, loz = (int)(bb.y & 0xffffu) << bsh;
                    const int hix = min((int)(bb.y >> 16) << bsh, P.nx), hiy = min((int)(bb.z & 0xffffu) << bsh, P.ny),
                              hiz = min((int)(bb.z >> 16) << bsh, P.nz);
                    ncross += mcrt::box_jump(ix, iy, iz, tmx, tmy, tmz, t, px, py, pz, ivx, ivy, ivz, ux, uy, uz,
                                             stx, sty, stz, lox, loy, loz, hix, hiy, hiz);
                    escaped = ((unsigned)ix >= (unsigned)P.nx) | ((unsigned)iy >= (unsigned)P.ny) |
                              ((unsigned)iz >= (unsigned)P.nz);
                    if (MCRT_J_ONELOAD) {
                        // the landing brick's entry: whether it is empty as well and, if so, its box -- one load per jump
                        busy = false;
                        if (!escaped) { bb = ldg_table(P.vbox + brick_of(ix, iy, iz, nbx, nby, bsh)); busy = bb.w != 0u; }
                    } else
                    busy = !escaped && brick_empty(s_m0, brick_of(ix, iy, iz, nbx, nby, bsh));
                }
            } while (__popc(__ballot_sync(kFull, busy)) >= max(jmin, 1));
            if (act) {
                SF(F_T, slot) = t;
                SU(U_NCROSS, slot) = ncross;
                if (escaped) {
                    SU(U_DK, slot) = (SU(U_DK, slot) & 0x3fffffffu) | (K_ESCAPED << 30);
                } else {
                    SU(U_W0, slot) = pack_xyz(ix, iy, iz);
                    if (!busy) {
                        const uint32_t cidx = lin_index(ix, iy, iz, lpx, lpxy);
                        SF(F_CW, slot) = __longlong_as_double((long long)__ldg(P.cellw + (size_t)kCS * cidx));
                    }
                }
            }
            const bool mine = act && !busy;   // still jumping: stays in mJ
            mJ.remove(mine, slot);
            mEv.add(mine && escaped, slot);
            mFly.add(mine && !escaped, slot);
            __syncwarp();
        } else if (nevt > 0) {
            // =========================================================== E phase: one event per lane
            const int nev = min(nevt, 32);
            const bool act = lane < nev;
            const int slot = act ? mEv.nth(lane) : 0;
            uint32_t kind = act ? (SU(U_DK, slot) >> 30) : 3u;
            uint32_t d = SU(U_DK, slot) & 0x3fffffffu;
            unsigned long long pid = 0ull, hash = 0ull;
            uint32_t ncross = 0u, nsca = 0u, nabs = 0u, nint = 0u;
            int ix = 0, iy = 0, iz = 0, j = 0;
            double ux = 0.0, uy = 0.0, uz = 1.0;
            bool insub = false;                         // the event happened / the new flight starts inside sub-cube (sgx, sgy, sgz)
            int sgx = 0, sgy = 0, sgz = 0;
            if (act && kind != K_EMIT) {
                pid = (unsigned long long)__double_as_longlong(SF(F_PID, slot));
                if (RECORD) hash = (unsigned long long)__double_as_longlong(SF(F_HASH, slot));
                ncross = SU(U_NCROSS, slot); nsca = SU(U_NSCA, slot); nabs = SU(U_NABS, slot);
                const uint32_t w0 = SU(U_W0, slot);
                ix = unpack_x(w0); iy = unpack_y(w0); iz = unpack_z(w0);
                j = (int)(SU(U_W1, slot) & 0xffffu); nint = SU(U_W1, slot) >> 16;
                if (XTRA && P.subR) {       // (no carry-over on divided grids: the upper half of U_W1 is the sub-cube state)
                    insub = kind == K_INTERACT && (SU(U_W1, slot) & kSubOk) != 0u;
                    sgx = (int)(nint & 7u); sgy = (int)((nint >> 3) & 7u); sgz = (int)((nint >> 6) & 7u);
                    nint = 0u;
                }
                ux = SF(F_UX, slot); uy = SF(F_UY, slot); uz = SF(F_UZ, slot);
                // per-cell redraw: the slot holds (index of the flight's draw) - (crossings at its start); every cell
                // entered since has used one more draw (see the walk), so the next free index is
                if (XTRA >= 3 && P.redraw) d = (d + ncross + 1u) & 0x3fffffffu;
            }
            {   // run counters of the packets that escape in this phase: summed over the warp, then added to the warp's
                // own counters in shared memory by one lane (no atomics)
                const bool esc = kind == K_ESCAPED;
                const unsigned em = __ballot_sync(kFull, esc);
                if (em) {
                    const uint32_t c_lo = __reduce_add_sync(kFull, esc ? (ncross & 0xffffu) : 0u);
                    const uint32_t c_hi = __reduce_add_sync(kFull, esc ? (ncross >> 16) : 0u);
                    const uint32_t n_sc = __reduce_add_sync(kFull, esc ? nsca : 0u);
                    const uint32_t n_ab = __reduce_add_sync(kFull, esc ? nabs : 0u);
                    const unsigned dm = __ballot_sync(kFull, esc && (nsca + nabs) == 0u);
                    if (lane == 0) {
                        volatile unsigned long long *wc = s_cnt + 8 * (threadIdx.x >> 5);
                        wc[CNT_PACKETS] += (unsigned long long)__popc(em);
                        wc[CNT_CROSS] += (unsigned long long)c_lo + ((unsigned long long)c_hi << 16);
                        wc[CNT_SCA] += (unsigned long long)n_sc;
                        wc[CNT_ABS] += (unsigned long long)n_ab;
                        wc[CNT_DIRECT] += (unsigned long long)__popc(dm);
                    }
                }
            }
            if (kind == K_ESCAPED) {
                // S10 escape tally: frequency x |cos i| bin, block-private histogram
                const double amu = fabs(uz);
                int bin = 0;
                for (int b = 1; b < P.ndir; ++b) if (s_mu[b] <= amu) bin = b;
                MCRT_CHK(bin >= 0 && bin < P.ndir && j >= 0 && j < nf, "escape: histogram bin");
                atomicAdd(&s_hist[bin * nf + j], 1u);
                const bool direct = (nsca + nabs) == 0u;
                if (direct) atomicAdd(&s_hist[P.ndir * nf + bin * nf + j], 1u);
                if (RECORD) {
                    hash_mix(hash, event_word(EV_ESCAPE, j, (unsigned long long)bin));
                    hash_mix(hash, (unsigned long long)ncross);
                    hash_mix(hash, (unsigned long long)nsca | ((unsigned long long)nabs << 32));
                    mcrt_digest dg;
                    dg.hash = hash; dg.crossings = ncross; dg.scatterings = nsca; dg.absorptions = nabs;
                    dg.escape_bin = (uint32_t)bin;
                    MCRT_CHK(pid - P.dig_base < P.dig_n, "escape: digest index");
                    P.dig[pid - P.dig_base] = dg;
                }
                kind = K_EMIT;        // the slot takes the next packet of the epoch
            }
            // S0 refill: the slots that need a new packet take the next ids with ONE atomic per warp
            const unsigned need = __ballot_sync(kFull, kind == K_EMIT);
            bool dead = false, resume = false;
            const unsigned long long n_take = P.count + (XTRA ? P.n_carry_in : 0u);   // carried packets first, then new ids
            uint32_t resume_idx = 0u;
            if (need) {
                unsigned long long base = n_take;
                if (!exhausted) {
                    const int leader = __ffs(need) - 1;
                    if (lane == leader) base = atomicAdd(&P.counters[CNT_NEXT], (unsigned long long)__popc(need));
                    base = __shfl_sync(kFull, base, leader);
                }
                if (kind == K_EMIT) {
                    const unsigned long long idx = base + (unsigned long long)__popc(need & ((1u << lane) - 1u));
                    if (XTRA && idx < P.n_carry_in) { resume = true; resume_idx = (uint32_t)idx; }
                    else if (idx < n_take) pid = P.pid0 + (idx - (XTRA ? P.n_carry_in : 0u));
                    else dead = true;
                }
                if (__any_sync(kFull, dead)) exhausted = true;   // the counter only grows
            }
            bool to_jump = false;                       // the new flight starts in an empty brick
            bool carried = false;                       // the packet's budget of this epoch is used up: carried over
            if (act && !dead) {
                double px, py, pz, z0, z1;
                bool scatter = false;
                double gmix = 0.0;                          // mixtures: g of the scattering component's material
                int sj = 0;
                unsigned long long cw;
                uint32_t cidx;
                if (XTRA && resume) {
                    // a packet carried over from the previous epoch: its state as it was left behind an interaction
                    const CarryRec rc = P.carry_in[resume_idx];
                    pid = rc.pid; hash = rc.hash; px = rc.px; py = rc.py; pz = rc.pz; ux = rc.ux; uy = rc.uy; uz = rc.uz;
                    ix = unpack_x(rc.w0); iy = unpack_y(rc.w0); iz = unpack_z(rc.w0);
                    j = (int)rc.j; d = rc.d; ncross = rc.ncross; nsca = rc.nsca; nabs = rc.nabs; nint = 0u;
                    cidx = lin_index(ix, iy, iz, lpx, lpxy);
                    to_jump = brick_empty(s_m0, brick_of(ix, iy, iz, nbx, nby, bsh));
                    cw = to_jump ? 0ull : __ldg(P.cellw + (size_t)kCS * cidx);
                } else if (kind == K_EMIT) {
                    // S2 emit: frequency through the source CDF (Eq. 1)
                    d = 0u; ncross = 0u; nsca = 0u; nabs = 0u; nint = 0u;
                    hash = 0xCBF29CE484222325ull;
                    draw2(P.seed_lo, P.seed_hi, pid, d++, P.pass, z0, z1);
                    // Eq. 1: stratified over the cumulative source spectrum, stratum = pid mod S
                    if (XTRA && P.source_strata) z0 = ((double)(pid % P.source_strata) + z0) / (double)P.source_strata;
                    j = lower_bound_cdf(s_src, nf, z0);
                    px = P.px; py = P.py; pz = P.pz;
                    cw = 0ull; cidx = 0u;
                } else {
                    // S5 partial segment up to the interaction point l' = tau/(rho kappa_ext) (Eq. 3)
                    px = SF(F_PX, slot); py = SF(F_PY, slot); pz = SF(F_PZ, slot);
                    const double t = SF(F_T, slot), tau = SF(F_TAU, slot), ztype = SF(F_ZTYPE, slot);
                    cw = (unsigned long long)__double_as_longlong(SF(F_CW, slot));
                    cidx = lin_index(ix, iy, iz, lpx, lpxy);
                    const double rho_c = cw_rho(cw);
                    sj = cw_species(cw) * nf + j;
                    const double2 kq = s_kk[sj];
                    const double kk = kq.x * rho_c;
                    const double sint = tau / kk;
                    const uint32_t hid = HOT ? cw_hot(cw, P.hot_shift, P.hot_mask) : 0u;
                    uint32_t fidx = 0u;                        // the sub-cube's index in the sub arrays
                    if (XTRA && insub) {
                        const unsigned long long pw = __ldg(P.cellw + (size_t)kCS * cidx);     // the divided cube's marker: its block
                        fidx = ((uint32_t)pw >> kSubShift) * (uint32_t)(P.subR * P.subR * P.subR) + (uint32_t)((sgz * P.subR + sgy) * P.subR + sgx);
                        lucy_add(P.sub_lfx, fidx, kq.y * rho_c * sint);
                    } else
                    if (hid) hot_add(s_hot, hid, lucy_round(kq.y * rho_c * sint));
                    else if (XTRA >= 2 && P.kmax_diag) {           // Sect. 3.1: Eq. 9, cells below the threshold only
                        if (rho_c * P.kmax_diag[cw_species(cw)] < kThinTau)
                            lucy_add(P.lfx, cidx, eq9_fx(kq.y * rho_c * sint, P.two_fx, P.inv_two_fx));
                    } else lucy_add(P.lfx, cidx, kq.y * rho_c * sint);
                    // mixtures (NEXT-3, readings Q34-Q36): the second component's tally; which component interacts
                    double2 thr = make_double2(2.0, 2.0);      // {S0, A0}; a uniform is < 2: one component = always component 0
                    if (XTRA >= 2 && P.lfx1) {
                        const double k1 = P.kabs1_fx[sj];
                        if (k1 != 0.0) lucy_add(P.lfx1, cidx, k1 * rho_c * sint);
                        if (P.mx_mat[2 * cw_species(cw) + 1] >= 0) thr = P.mx_thr[sj];
                    }
                    const double tint = t + sint;
                    double q;
                    if (XTRA && insub) {    // the interaction point stays inside its sub-cube
                        const double Rd = (double)P.subR;
                        q = px + ux * tint; q = fmax(q, (double)ix + (double)sgx / Rd); q = fmin(q, (double)ix + (double)(sgx + 1) / Rd); px = q;
                        q = py + uy * tint; q = fmax(q, (double)iy + (double)sgy / Rd); q = fmin(q, (double)iy + (double)(sgy + 1) / Rd); py = q;
                        q = pz + uz * tint; q = fmax(q, (double)iz + (double)sgz / Rd); q = fmin(q, (double)iz + (double)(sgz + 1) / Rd); pz = q;
                    } else {
                    q = px + ux * tint; q = fmax(q, (double)ix); q = fmin(q, (double)(ix + 1)); px = q;
                    q = py + uy * tint; q = fmax(q, (double)iy); q = fmin(q, (double)(iy + 1)); py = q;
                    q = pz + uz * tint; q = fmax(q, (double)iz); q = fmin(q, (double)(iz + 1)); pz = q;
                    }
                    const unsigned long long cell = (XTRA && insub) ? P.nc_grid + fidx : ((unsigned long long)iz * P.ny + iy) * P.nx + ix;
                    // S6 scatter with probability albedo
                    if (ztype < s_ag[sj].x) {
                        scatter = true;
                        nsca++;
                        if (XTRA && P.sca_slot && P.sca_slot[j] >= 0) {   // store the event: cell, frequency, incoming direction
                            const unsigned long long at = atomicAdd(&P.counters[CNT_SCAEV], 1ull);
                            if (at < P.sca_cap) {
                                mcrt_scatter_event ev;
                                ev.cell = (uint32_t)cell; ev.slot = (uint16_t)P.sca_slot[j];
                                ev.q[0] = (int16_t)__double2ll_rn(32767.0 * ux);
                                ev.q[1] = (int16_t)__double2ll_rn(32767.0 * uy);
                                ev.q[2] = (int16_t)__double2ll_rn(32767.0 * uz);
                                P.sca_ev[at] = ev;
                            }
                        }
                        if (RECORD) hash_mix(hash, event_word(EV_SCATTER, j, cell));
                        if (XTRA >= 2 && P.lfx1) gmix = P.g[P.mx_mat[2 * cw_species(cw) + (!(ztype < thr.x) ? 1 : 0)] * nf + j];
                    } else {
                        // S8/S9 absorb: count, re-emit at once at a frequency drawn from the
                        // cell's frozen-epoch temperature row of Eq. 10 or Eq. 5 (sweeps)
                        nabs++;
                        MCRT_CHK(cidx < P.ncp, "absorption: storage index of the cell");
                        int s = cw_species(cw);
                        int m = cw_tidx(cw, P.tidx_mask);
                        bool second = false;                   // absorbed by the second component of a mixture
                        if (XTRA >= 2 && P.lfx1) {
                            second = !(ztype < thr.y);
                            s = P.mx_mat[2 * s + (second ? 1 : 0)];    // the material whose row re-emits
                            if (second) m = (int)P.tidx1[cidx];
                        }
                        if (XTRA && P.live_bw) {
                            // Bjorkman & Wood as printed: the temperature is adjusted after each
                            // absorption -- T_{i,k} from the count including this one (Eq. 4).  The count a packet sees
                            // depends on the order of the atomics: results are reproducible only statistically.
                            const unsigned long long kn = atomicAdd(&P.kcnt[cidx], 1ull) + 1ull;
                            m = t_index(P.J + s * P.nT, P.nT, (double)kn * P.cellfac / rho_c);
                        } else if (XTRA && insub) atomicAdd(&P.sub_kcnt[fidx], 1ull);
                        else if (hid) atomicAdd(&s_hot[3u * hid + 2u], 1u);
                        else if (XTRA >= 2 && second) atomicAdd(&P.kcnt1[cidx], 1ull);
                        else atomicAdd(&P.kcnt[cidx], 1ull);
                        draw2(P.seed_lo, P.seed_hi, pid, d++, P.pass, z0, z1);
                        MCRT_CHK(s >= 0 && s < P.ns && m >= 0 && m < P.nT, "absorption: CDF row");
                        j = lower_bound_eytzinger(P.cdf + ((size_t)s * P.nT + m) * P.nfs, nf < kPermSmem ? s_perm : P.perm, nf, z0);
                        if (RECORD) hash_mix(hash, event_word(EV_ABSORB, j, cell));
                    }
                }
                if (!(XTRA && resume)) {
                // new direction: isotropic or Henyey-Greenstein about the old one (S7)
                draw2(P.seed_lo, P.seed_hi, pid, d++, P.pass, z0, z1);
                double mu = 1.0 - 2.0 * z0;
                if (scatter) {
                    const double gg = (XTRA >= 2 && P.lfx1) ? gmix : s_ag[sj].y;
                    if (fabs(gg) > 1e-6) {
                        const double q = (1.0 - gg * gg) / (1.0 - gg + 2.0 * gg * z0);
                        mu = (1.0 + gg * gg - q * q) / (2.0 * gg);
                        mu = fmin(mu, 1.0);
                        mu = fmax(mu, -1.0);
                    }
                }
                double sp, cp;
                traj_sincos_turns(z1, sp, cp);   // phi = 2 pi z1
                const double st = sqrt(1.0 - mu * mu);
                if (scatter) {
                    double a0, a1, a2;
                    if (fabs(uz) > 0.99999) {
                        a0 = st * cp;
                        a1 = st * sp;
                        a2 = (uz > 0.0) ? mu : -mu;
                    } else {
                        const double w = sqrt(1.0 - uz * uz);
                        const double iw = 1.0 / w;
                        const double t0 = ux * uz * cp - uy * sp;
                        const double t1 = uy * uz * cp + ux * sp;
                        a0 = st * t0 * iw + ux * mu;
                        a1 = st * t1 * iw + uy * mu;
                        a2 = uz * mu - st * cp * w;
                    }
                    const double inorm = 1.0 / sqrt(a0 * a0 + a1 * a1 + a2 * a2);
                    ux = a0 * inorm; uy = a1 * inorm; uz = a2 * inorm;
                } else {
                    ux = st * cp; uy = st * sp; uz = mu;
                }
                if (kind == K_EMIT) {
                    // start cell: floor(p), or by direction sign when p sits on a face (reading Q9)
                    double f;
                    f = floor(px); ix = (px != f) ? (int)f : ((ux >= 0.0) ? (int)f : (int)f - 1);
                    f = floor(py); iy = (py != f) ? (int)f : ((uy >= 0.0) ? (int)f : (int)f - 1);
                    f = floor(pz); iz = (pz != f) ? (int)f : ((uz >= 0.0) ? (int)f : (int)f - 1);
                    const uint32_t brick = brick_of(ix, iy, iz, nbx, nby, bsh);
                    cidx = lin_index(ix, iy, iz, lpx, lpxy);
                    to_jump = brick_empty(s_m0, brick);
                    cw = to_jump ? 0ull : __ldg(P.cellw + (size_t)kCS * cidx);
                    if (XTRA && P.subR && (uint32_t)(cw >> 32) == kMarkHi && ((uint32_t)cw & kSubFlag)) {
                        // the source stands in a divided cube: the same start rule on the lattice of sub-cube faces
                        const double Rd = (double)P.subR;
                        double pf;
                        pf = px * Rd; f = floor(pf); sgx = ((pf != f) ? (int)f : ((ux >= 0.0) ? (int)f : (int)f - 1)) - ix * P.subR;
                        pf = py * Rd; f = floor(pf); sgy = ((pf != f) ? (int)f : ((uy >= 0.0) ? (int)f : (int)f - 1)) - iy * P.subR;
                        pf = pz * Rd; f = floor(pf); sgz = ((pf != f) ? (int)f : ((uz >= 0.0) ? (int)f : (int)f - 1)) - iz * P.subR;
                        insub = true;
                    }
                    if (RECORD)
                        hash_mix(hash, event_word(EV_EMIT, j, ((unsigned long long)iz * P.ny + iy) * P.nx + ix));
                } else if (XTRA && P.carry_K && ++nint >= P.carry_K) {
                    // carry-over: the interaction budget of this epoch is used up.  The packet's state goes to the
                    // list the next epoch starts with; the slot takes another packet.
                    carried = true;
                    CarryRec rc;
                    rc.pid = pid; rc.hash = hash; rc.px = px; rc.py = py; rc.pz = pz; rc.ux = ux; rc.uy = uy; rc.uz = uz;
                    rc.w0 = pack_xyz(ix, iy, iz); rc.j = (uint32_t)j; rc.d = d; rc.ncross = ncross; rc.nsca = nsca; rc.nabs = nabs;
                    P.carry_out[atomicAdd(&P.counters[CNT_CARRY], 1ull)] = rc;
                    SU(U_DK, slot) = K_EMIT << 30;
                }
                }   // !resume
                if (!carried) {
                // S3 optical depth of the flight: tau = -ln zeta, zeta_1 kept for S6
                draw2(P.seed_lo, P.seed_hi, pid, d++, P.pass, z0, z1);
                // park the new flight (reading Q8: the walk needs p, 1/u, the cell; t = 0)
                SF(F_PX, slot) = px; SF(F_PY, slot) = py; SF(F_PZ, slot) = pz;
                SF(F_UX, slot) = ux; SF(F_UY, slot) = uy; SF(F_UZ, slot) = uz;
#if MCRT_SLOT_IV
                SF(F_IVX, slot) = (ux != 0.0) ? 1.0 / ux : CUDART_INF;
                SF(F_IVY, slot) = (uy != 0.0) ? 1.0 / uy : CUDART_INF;
                SF(F_IVZ, slot) = (uz != 0.0) ? 1.0 / uz : CUDART_INF;
#endif
                SF(F_T, slot) = 0.0;
                SF(F_TAU, slot) = -traj_log(z0);
                SF(F_ZTYPE, slot) = z1;
                SF(F_CW, slot) = __longlong_as_double((long long)cw);
                SF(F_PID, slot) = __longlong_as_double((long long)pid);
                if (RECORD) SF(F_HASH, slot) = __longlong_as_double((long long)hash);
                // (kind is set when the walk stops.)  Per-cell redraw: the cell reached after c crossings of
                // this flight takes the draw of index (flight's draw) + c -- c = 0 is the flight's own draw, so the first
                // cell needs no special case -- and the slot keeps that index minus the crossing count
                SU(U_DK, slot) = (XTRA >= 3 && P.redraw) ? ((d - 1u - ncross) & 0x3fffffffu) : d;
                SU(U_NCROSS, slot) = ncross; SU(U_NSCA, slot) = nsca; SU(U_NABS, slot) = nabs;
                SU(U_W0, slot) = pack_xyz(ix, iy, iz);
                SU(U_W1, slot) = (uint32_t)j | (nint << 16) | ((XTRA && insub) ? sub_pack(sgx, sgy, sgz) : 0u);
                }   // !carried
            }
            mEv.remove(act && !carried, slot);             // taken: now flying, jumping, or dead (no packets left)
            const bool to_sub = XTRA && insub && act && !dead && !carried;      // the new flight starts inside a sub-cube
            if (XTRA) mSub.add(to_sub, slot);
            mFly.add(act && !dead && !to_jump && !carried && !to_sub, slot);
            mJ.add(act && !dead && to_jump && !carried, slot);
            __syncwarp();
        } else {
            break;
        }
    }
#undef SF
#undef SU
    {   // dusty crossings stepped by this warp
        const uint32_t nd = __reduce_add_sync(kFull, ndusty_acc & 0xffffu), ndh = __reduce_add_sync(kFull, ndusty_acc >> 16);
        if (lane == 0) s_cnt[8 * (threadIdx.x >> 5) + CNT_DUSTY] += (unsigned long long)nd + ((unsigned long long)ndh << 16);
    }

    // flush the block-private histogram and counters
    __syncthreads();
    if (HOT)
        for (int i = 1 + (int)threadIdx.x; i <= P.n_hot; i += blockDim.x) {
            const unsigned long long v = ((unsigned long long)s_hot[3 * i + 1] << 32) + s_hot[3 * i];
            const uint32_t ci = P.hot_idx[i];
            if (v) lucy_add_raw(P.lfx, ci, v);
            if (s_hot[3 * i + 2]) atomicAdd(&P.kcnt[ci], (unsigned long long)s_hot[3 * i + 2]);
        }
    const int half = P.ndir * nf;
    for (int i = threadIdx.x; i < nhist; i += blockDim.x) {
        const unsigned int v = s_hist[i];
        if (v) atomicAdd(i < half ? &P.sed[i] : &P.sed_direct[i - half], (unsigned long long)v);
    }
    if (threadIdx.x < CNT_NEXT && threadIdx.x != CNT_OVERFLOW) {
        unsigned long long v = 0ull;
        for (int w = 0; w < nwarps; ++w) v += s_cnt[8 * w + threadIdx.x];
        if (v) atomicAdd(&P.counters[threadIdx.x], v);
    }
}

// ------------------------------------------------------------------------------------------------
// S11 epoch temperature-index update (streaming over cells, between transport launches).
//   k~ = k + max(1, 1/2 (k - k_prev) B_e/B_{e-1});  x = k~ xi / (4 pi rho h^3) (Eq. 4);
//   tidx = #{ J[s][.] < x } clamped to [0, nT-1];  k_prev = k.   Also checks the fixed-point range.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int t_index(const double *J, int nT, double x)
{
    int lo = 0, hi = nT;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (J[mid] < x) lo = mid + 1; else hi = mid;
    }
    return lo > nT - 1 ? nT - 1 : lo;
}

__global__ void __launch_bounds__(256) k_epoch_update(unsigned long long *__restrict__ cellw, const unsigned long long *__restrict__ kcnt,
                                                      unsigned long long *__restrict__ kprev,
                                                      const long long *__restrict__ lfx, const double *__restrict__ J,
                                                      int nT, int ns, size_t ncp, int first_epoch, double ratio,
                                                      double cellfac, unsigned long long *__restrict__ counters, uint32_t tmask)
{
    extern __shared__ double s_J[];
    for (int i = threadIdx.x; i < ns * nT; i += blockDim.x) s_J[i] = J[i];
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) { counters[CNT_NEXT] = 0ull; counters[CNT_CARRY] = 0ull; }
    bool ovf = false;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncp; i += (size_t)gridDim.x * blockDim.x) {
        const unsigned long long cw = cellw[kCS * i];
        const double rho_c = cw_rho(cw);
        const unsigned long long kc = kcnt[i];
        uint32_t m = 0u;
        if (cw_dusty(cw)) {
            double kt;
            if (first_epoch) kt = (double)kc + 1.0;
            else {
                const double pred = 0.5 * (double)(kc - kprev[i]) * ratio;
                kt = (double)kc + ((pred > 1.0) ? pred : 1.0);
            }
            const double x = kt * cellfac / rho_c;
            m = (uint32_t)t_index(s_J + cw_species(cw) * nT, nT, x);
            const long long v = lfx[kCS * i];
            ovf |= (v > (1ll << 62)) || (v < -(1ll << 62));
        }
        kprev[i] = kc;
        const uint32_t lo = (uint32_t)cw, nlo = (lo & ~(tmask << 8)) | (m << 8);
        // low word: species | tidx << 8 | hot number | rho bits 29-31 (the words of vacuum and marker cells are never written)
        if (nlo != lo && cw_dusty(cw)) reinterpret_cast<uint32_t *>(cellw + kCS * i)[0] = nlo;
    }
    if (ovf) counters[CNT_OVERFLOW] = 1ull;
}

// S12 temperature index for a frozen-T sweep from the previous pass's tallies; zeroes them.
__global__ void __launch_bounds__(256) k_sweep_update(unsigned long long *__restrict__ cellw, unsigned long long *__restrict__ kcnt,
                                                      unsigned long long *__restrict__ kprev, long long *__restrict__ lfx,
                                                      const double *__restrict__ J, int nT, int ns, size_t ncp,
                                                      int from_lucy, double inv_fx, double cellfac,
                                                      unsigned long long *__restrict__ counters, uint32_t tmask)
{
    extern __shared__ double s_J[];
    for (int i = threadIdx.x; i < ns * nT; i += blockDim.x) s_J[i] = J[i];
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) counters[CNT_NEXT] = 0ull;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncp; i += (size_t)gridDim.x * blockDim.x) {
        const unsigned long long cw = cellw[kCS * i];
        const double rho_c = cw_rho(cw);
        uint32_t m = 0u;
        if (cw_dusty(cw)) {
            const double e = from_lucy ? (double)lfx[kCS * i] * inv_fx : (double)kcnt[i];
            const double x = e * cellfac / rho_c;
            m = (uint32_t)t_index(s_J + cw_species(cw) * nT, nT, x);
        }
        if (cw_dusty(cw)) reinterpret_cast<uint32_t *>(cellw + kCS * i)[0] = ((uint32_t)cw & ~(tmask << 8)) | (m << 8);
        kcnt[i] = 0ull;
        kprev[i] = 0ull;
        lfx[kCS * i] = 0ll;
    }
}

// The same two updates for a grid of dust mixtures (NEXT-3; reading Q36): every component has its own count, tally
// and temperature index -- Eq. 4 with the component's material and its own mass rho f_c V.  Component 0's index
// lives in the cell word, component 1's in tidx1.  sweep = 0: epoch rule (S11), 1: frozen-T sweep (S12, zeroes the tallies).
struct MixArrays {
    unsigned long long *kcnt[2], *kprev[2];
    long long *lfx[2];
    uint16_t *tidx1;
    const int *ncomp, *mat;
    const double *frac;
};
__global__ void __launch_bounds__(256) k_mix_update(unsigned long long *__restrict__ cellw, MixArrays A, const double *__restrict__ J,
                                                    int nT, int ns, size_t ncp, int sweep, int first_epoch, double ratio,
                                                    int from_lucy, double inv_fx, double cellfac,
                                                    unsigned long long *__restrict__ counters, uint32_t tmask)
{
    extern __shared__ double s_J[];
    for (int i = threadIdx.x; i < ns * nT; i += blockDim.x) s_J[i] = J[i];
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) { counters[CNT_NEXT] = 0ull; if (!sweep) counters[CNT_CARRY] = 0ull; }
    bool ovf = false;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncp; i += (size_t)gridDim.x * blockDim.x) {
        const unsigned long long cw = cellw[kCS * i];
        const double rho_c = cw_rho(cw);
        const bool dusty = cw_dusty(cw);
        const int x = (int)cw_species(cw);
        uint32_t mi[2] = {0u, 0u};
        for (int c = 0; c < 2; ++c) {
            const unsigned long long kc = A.kcnt[c][i];
            if (dusty && c < A.ncomp[x]) {
                const long long v = A.lfx[c][kCS * i];
                double e;
                if (sweep) e = from_lucy ? (double)v * inv_fx : (double)kc;
                else if (first_epoch) e = (double)kc + 1.0;
                else {
                    const double pred = 0.5 * (double)(kc - A.kprev[c][i]) * ratio;
                    e = (double)kc + ((pred > 1.0) ? pred : 1.0);
                }
                const double xx = e * cellfac / (rho_c * A.frac[2 * x + c]);
                mi[c] = (uint32_t)t_index(s_J + A.mat[2 * x + c] * nT, nT, xx);
                ovf |= (v > (1ll << 62)) || (v < -(1ll << 62));
            }
            if (sweep) { A.kcnt[c][i] = 0ull; A.kprev[c][i] = 0ull; A.lfx[c][kCS * i] = 0ll; }
            else A.kprev[c][i] = kc;
        }
        const uint32_t lo = (uint32_t)cw, nlo = (lo & ~(tmask << 8)) | (mi[0] << 8);
        if (nlo != lo && dusty) reinterpret_cast<uint32_t *>(cellw + kCS * i)[0] = nlo;
        A.tidx1[i] = (uint16_t)mi[1];
    }
    if (ovf && !sweep) counters[CNT_OVERFLOW] = 1ull;
}

// The two updates under the thresholded estimator of Sect. 3.1 (reading Q39): a cell below the threshold takes its
// temperature from its Eq. 9 energy (the same midpoint prediction, on the tally; k_prev keeps the tally there), every
// other cell from its count as above.  sweep = 0: epoch rule (S11), 1: frozen-T sweep (S12, zeroes the tallies).
__global__ void __launch_bounds__(256) k_hybrid_update(unsigned long long *__restrict__ cellw, unsigned long long *__restrict__ kcnt,
                                                       unsigned long long *__restrict__ kprev, long long *__restrict__ lfx,
                                                       const double *__restrict__ J, const double *__restrict__ kmax_diag, int nT,
                                                       int ns, size_t ncp, int sweep, int first_epoch, double ratio, double inv_fx,
                                                       double cellfac, unsigned long long *__restrict__ counters, uint32_t tmask)
{
    extern __shared__ double s_J[];
    for (int i = threadIdx.x; i < ns * nT; i += blockDim.x) s_J[i] = J[i];
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) { counters[CNT_NEXT] = 0ull; if (!sweep) counters[CNT_CARRY] = 0ull; }
    bool ovf = false;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncp; i += (size_t)gridDim.x * blockDim.x) {
        const unsigned long long cw = cellw[kCS * i];
        const double rho_c = cw_rho(cw);
        const unsigned long long kc = kcnt[i];
        const long long v = lfx[kCS * i];
        uint32_t m = 0u;
        bool thin = false;
        if (cw_dusty(cw)) {
            thin = rho_c * kmax_diag[cw_species(cw)] < kThinTau;
            double e;
            if (thin) {
                const double E = (double)v * inv_fx, Ep = (double)(long long)kprev[i] * inv_fx;
                e = (sweep || first_epoch) ? E : E + 0.5 * (E - Ep) * ratio;
            } else if (sweep) e = (double)kc;
            else if (first_epoch) e = (double)kc + 1.0;
            else {
                const double pred = 0.5 * (double)(kc - kprev[i]) * ratio;
                e = (double)kc + ((pred > 1.0) ? pred : 1.0);
            }
            m = (uint32_t)t_index(s_J + cw_species(cw) * nT, nT, e * cellfac / rho_c);
            ovf |= (v > (1ll << 62)) || (v < -(1ll << 62));
        }
        if (sweep) { kcnt[i] = 0ull; kprev[i] = 0ull; lfx[kCS * i] = 0ll; }
        else kprev[i] = thin ? (unsigned long long)v : kc;
        const uint32_t lo = (uint32_t)cw, nlo = (lo & ~(tmask << 8)) | (m << 8);
        if (nlo != lo && cw_dusty(cw)) reinterpret_cast<uint32_t *>(cellw + kCS * i)[0] = nlo;
    }
    if (ovf && !sweep) counters[CNT_OVERFLOW] = 1ull;
}

// Partitioned runs: between epochs a part's absorption counts are exchanged as this epoch's own
// increments, k - k_prev (k_prev = the global counts at the start of the epoch), and restored afterwards.
__global__ void __launch_bounds__(256) k_count_delta(unsigned long long *__restrict__ kcnt, const unsigned long long *__restrict__ kprev,
                                                     size_t n, int restore)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        kcnt[i] = restore ? kcnt[i] + kprev[i] : kcnt[i] - kprev[i];
}

// gathers the Lucy tallies (stride kCS) into a contiguous buffer for the exchange, and back
__global__ void __launch_bounds__(256) k_lucy_stage(long long *__restrict__ lfx, long long *__restrict__ stage, size_t n, int back)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        if (back) lfx[kCS * i] = stage[i]; else stage[i] = lfx[kCS * i];
    }
}

// Sum of the parts' tallies over peer-visible memory, reduce-scatter / all-gather (mcrt_exchange_peer_sum):
// phase 0: own[i] = sum_p part_p[i] for i in this part's slice; phase 1: own[i] = owner(i)[i] for the other slices.
constexpr int kMaxParts = 16;
struct PeerPtrs { unsigned long long *p[kMaxParts]; };
__global__ void __launch_bounds__(256) k_peer_sum(PeerPtrs pp, int me, int n_parts, size_t words, int phase)
{
    const size_t per = (words + (size_t)n_parts - 1) / (size_t)n_parts;
    if (phase == 0) {
        const size_t lo = per * (size_t)me, hi = lo + per < words ? lo + per : words;
        for (size_t i = lo + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < hi; i += (size_t)gridDim.x * blockDim.x) {
            unsigned long long v = 0ull;
            for (int q = 0; q < n_parts; ++q) v += pp.p[q][i];
            pp.p[me][i] = v;
        }
    } else {
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < words; i += (size_t)gridDim.x * blockDim.x) {
            const int owner = (int)(i / per);
            if (owner != me) pp.p[me][i] = pp.p[owner][i];
        }
    }
}

// range check of the fixed-point tallies after the last epoch (|L| <= 2^62, O9)
__global__ void __launch_bounds__(256) k_range_check(const long long *__restrict__ lfx, size_t ncp,
                                                     unsigned long long *__restrict__ counters)
{
    bool ovf = false;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncp; i += (size_t)gridDim.x * blockDim.x) {
        const long long v = lfx[kCS * i];
        ovf |= (v > (1ll << 62)) || (v < -(1ll << 62));
    }
    if (ovf) counters[CNT_OVERFLOW] = 1ull;
}

// ------------------------------------------------------------------------------------------------
// layout kernels: canonical [nz][ny][nx] <-> brick-major
// ------------------------------------------------------------------------------------------------
__global__ void k_pack_grid(const float *__restrict__ rho, const uint8_t *__restrict__ sp, unsigned long long *__restrict__ cellw,
                            int nx, int ny, int nz, int px, int pxy, size_t ncp, int ns, unsigned long long *__restrict__ bad)
{
    for (size_t b = (size_t)blockIdx.x * blockDim.x + threadIdx.x; b < ncp; b += (size_t)gridDim.x * blockDim.x) {
        const int iz = (int)(b / (size_t)pxy) - kGuard;
        const int rem = (int)(b % (size_t)pxy);
        const int iy = rem / px - kGuard, ix = rem % px - kGuard;
        unsigned long long cw = kOutWord;        // the guard shell: "outside the grid"
        if ((unsigned)ix < (unsigned)nx && (unsigned)iy < (unsigned)ny && (unsigned)iz < (unsigned)nz) {
            const size_t i = ((size_t)iz * ny + iy) * nx + ix;
            const float r = rho[i];
            const uint32_t s = sp[i];
            if (!(r >= 0.0f) || isinf(r)) atomicAdd(&bad[0], 1ull);
            if (s >= (uint32_t)ns) atomicAdd(&bad[1], 1ull);
            // fp32 -> fp64 is exact and leaves the low 29 mantissa bits zero; -0 is stored as +0
            const double rd = (r > 0.0f && !isinf(r)) ? (double)r : 0.0;
            if (rd > 0.0) atomicAdd(&bad[2], 1ull);   // number of dusty cells (chooses the walk variant)
            cw = ((unsigned long long)__double_as_longlong(rd) & kRhoMask) | (unsigned long long)(s & 0xffu);
        }
        cellw[kCS * b] = cw;
    }
}

// mcrt_subgrid: packs the sub-cubes' cell words and turns the divided cubes' words into markers with their block number.
// bad[0] counts divided cubes whose own density is not > 0 (their brick would count as empty), bad[1] bad sub-cubes.
__global__ void k_pack_sub(unsigned long long *__restrict__ cellw, unsigned long long *__restrict__ sub_cellw,
                           const long long *__restrict__ cube, const float *__restrict__ rho, const uint8_t *__restrict__ sp,
                           size_t n_sub, int R3, int nx, int ny, int nz, int px, int pxy, int ns, unsigned long long *__restrict__ bad)
{
    const size_t n = n_sub * (size_t)R3;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float r = rho[i];
        const uint32_t s = sp[i];
        if (!(r >= 0.0f) || isinf(r) || s >= (uint32_t)ns) atomicAdd(&bad[1], 1ull);
        const double rd = (r > 0.0f && !isinf(r)) ? (double)r : 0.0;
        sub_cellw[kCS * i] = ((unsigned long long)__double_as_longlong(rd) & kRhoMask) | (unsigned long long)(s & 0xffu);
        if (i % (size_t)R3 == 0) {
            const size_t b = i / (size_t)R3;
            const long long ci = cube[b];
            const int ix = (int)(ci % nx), iy = (int)((ci / nx) % ny), iz = (int)(ci / ((long long)nx * ny));
            unsigned long long *w = cellw + (size_t)kCS * lin_index(ix, iy, iz, px, pxy);
            if (!cw_dusty(*w)) atomicAdd(&bad[0], 1ull);
            *w = kJumpWord | kSubFlag | ((unsigned long long)b << kSubShift);
        }
    }
}

// the outputs of mcrt_read / mcrt_read_raw for the sub-cubes (identity order; Eq. 4 with V = (h/R)^3 through cellfac)
__global__ void k_gather_sub(int what, void *__restrict__ out, const unsigned long long *__restrict__ cellw,
                             const unsigned long long *__restrict__ kcnt, const long long *__restrict__ lfx,
                             const double *__restrict__ J, const double *__restrict__ Tg, int nT, size_t off, size_t n, double xi,
                             double inv_fx, double cellfac, uint32_t tmask);

// The species byte of a vacuum cell means nothing (rho = 0 makes every product of the walk 0), but the walk reloads its
// cached opacities whenever the byte changes.  So a vacuum cell inside a dusty brick takes the species of the nearest
// dusty cell along the axes (fixed search order, up to kVacReach cells: deterministic; only dusty cells are read for
// their species and those are never written): a ray that leaves a clump, crosses a gap and enters the next reloads
// once instead of twice.  Run after k_build_mask0 (the cells of empty bricks are marker words by then and stay).
constexpr int kVacReach = 4;
__global__ void k_vac_species(unsigned long long *__restrict__ cellw, int nx, int ny, int nz, int px, int pxy)
{
    const size_t nc = (size_t)nx * ny * nz;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nc; i += (size_t)gridDim.x * blockDim.x) {
        const int ix = (int)(i % nx), iy = (int)((i / nx) % ny), iz = (int)(i / ((size_t)nx * ny));
        const size_t b = lin_index(ix, iy, iz, px, pxy);
        const unsigned long long cw = cellw[kCS * b];
        if ((cw >> 32) != 0ull) continue;                    // dusty or marker
        const int step[6] = {-1, 1, -px, px, -pxy, pxy};
        const int room[6] = {ix, nx - 1 - ix, iy, ny - 1 - iy, iz, nz - 1 - iz};
        int found = -1;
        for (int d = 1; d <= kVacReach && found < 0; ++d)
            for (int a = 0; a < 6 && found < 0; ++a) {
                if (d > room[a]) continue;
                const unsigned long long w = cellw[kCS * (size_t)((long long)b + (long long)d * step[a])];
                if (cw_dusty(w)) found = (int)cw_species(w);
            }
        if (found >= 0 && (uint32_t)found != cw_species(cw))
            reinterpret_cast<uint32_t *>(cellw + kCS * b)[0] = ((uint32_t)cw & ~0xffu) | (uint32_t)found;
    }
}

// Vacuum mask of one level: bit of box (bx, by, bz) is set when all its in-grid cells have rho == 0.
// Level 0 is built from the packed cells, level l > 0 from level l - 1 (4x4x4 children per box).
__global__ void k_build_mask0(unsigned long long *__restrict__ cellw, uint32_t *__restrict__ m, int nx, int ny, int nz,
                              int px, int pxy, int sh, int mbx, int mby, int mbz)
{
    const int nb = mbx * mby * mbz;
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < nb; b += gridDim.x * blockDim.x) {
        const int bx = b % mbx, by = (b / mbx) % mby, bz = b / (mbx * mby);
        const int x0 = bx << sh, y0 = by << sh, z0 = bz << sh;
        const int x1 = min(x0 + (1 << sh), nx), y1 = min(y0 + (1 << sh), ny), z1 = min(z0 + (1 << sh), nz);
        bool empty = true;
        for (int z = z0; z < z1 && empty; ++z)
            for (int y = y0; y < y1 && empty; ++y)
                for (int x = x0; x < x1; ++x)
                    if (!cw_vacuum(cellw[(size_t)kCS * lin_index(x, y, z, px, pxy)])) { empty = false; break; }
        if (empty) {
            atomicOr(&m[b >> 5], 1u << (b & 31));
            // every cell word of an empty brick carries the marker bit: the cell walk sees it in the word it reads
            // anyway and needs no mask lookup
            for (int z = z0; z < z1; ++z)
                for (int y = y0; y < y1; ++y)
                    for (int x = x0; x < x1; ++x) cellw[(size_t)kCS * lin_index(x, y, z, px, pxy)] |= kJumpWord;
        }
    }
}

// Empty boxes for the J phase.  sat[z][y][x] (dims nb+1) = number of dusty bricks in [0,x) x [0,y) x [0,z): built
// by three prefix passes; k_grow_boxes then grows, for every empty brick, a box of empty bricks around it: the
// six faces are pushed out one layer at a time, round robin, as long as the added layer holds no dust (one
// summed-area query each), so the box first grows like a cube and then keeps extending where space is left.
__global__ void k_sat_pass(const uint32_t *__restrict__ mask, int *__restrict__ sat, int nbx, int nby, int nbz, int axis)
{
    const int sx = nbx + 1, sy = nby + 1;
    const int n1 = axis == 0 ? nby : nbx, n2 = axis == 2 ? nby : nbz;   // the two axes a thread does not scan
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n1 * n2; i += gridDim.x * blockDim.x) {
        const int a = i % n1, b = i / n1;
        int run = 0;
        if (axis == 0) {
            for (int x = 0; x < nbx; ++x) {
                const int o = (b * nby + a) * nbx + x;
                run += ((mask[o >> 5] >> (o & 31)) & 1u) ? 0 : 1;
                sat[((size_t)(b + 1) * sy + (a + 1)) * sx + (x + 1)] = run;
            }
        } else if (axis == 1) {
            for (int y = 0; y < nby; ++y) {
                int *q = sat + ((size_t)(b + 1) * sy + (y + 1)) * sx + (a + 1);
                run += *q; *q = run;
            }
        } else {
            for (int z = 0; z < nbz; ++z) {
                int *q = sat + ((size_t)(z + 1) * sy + (b + 1)) * sx + (a + 1);
                run += *q; *q = run;
            }
        }
    }
}

__device__ __forceinline__ int sat_count(const int *__restrict__ sat, int sx, int sy, int x0, int y0, int z0, int x1, int y1, int z1)
{
#define SAT_(x, y, z) sat[((size_t)(z) * sy + (y)) * sx + (x)]
    return SAT_(x1, y1, z1) - SAT_(x0, y1, z1) - SAT_(x1, y0, z1) - SAT_(x1, y1, z0) + SAT_(x0, y0, z1) + SAT_(x0, y1, z0) +
           SAT_(x1, y0, z0) - SAT_(x0, y0, z0);
#undef SAT_
}

__global__ void k_grow_boxes(const uint32_t *__restrict__ mask, const int *__restrict__ sat, uint4 *__restrict__ box, int nbx,
                             int nby, int nbz)
{
    const int nb = nbx * nby * nbz, sx = nbx + 1, sy = nby + 1;
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < nb; b += gridDim.x * blockDim.x) {
        int x0 = b % nbx, y0 = (b / nbx) % nby, z0 = b / (nbx * nby);
        int x1 = x0 + 1, y1 = y0 + 1, z1 = z0 + 1;
        if ((mask[b >> 5] >> (b & 31)) & 1u) {
            bool grew = true;
            while (grew) {
                grew = false;
                if (x0 > 0 && sat_count(sat, sx, sy, x0 - 1, y0, z0, x0, y1, z1) == 0) { --x0; grew = true; }
                if (x1 < nbx && sat_count(sat, sx, sy, x1, y0, z0, x1 + 1, y1, z1) == 0) { ++x1; grew = true; }
                if (y0 > 0 && sat_count(sat, sx, sy, x0, y0 - 1, z0, x1, y0, z1) == 0) { --y0; grew = true; }
                if (y1 < nby && sat_count(sat, sx, sy, x0, y1, z0, x1, y1 + 1, z1) == 0) { ++y1; grew = true; }
                if (z0 > 0 && sat_count(sat, sx, sy, x0, y0, z0 - 1, x1, y1, z0) == 0) { --z0; grew = true; }
                if (z1 < nbz && sat_count(sat, sx, sy, x0, y0, z1, x1, y1, z1 + 1) == 0) { ++z1; grew = true; }
            }
        }
        // (fourth word: 1 = the brick is empty -- the jump loop reads "is the landing brick empty" and its box in one load)
        box[b] = make_uint4((uint32_t)x0 | ((uint32_t)y0 << 16), (uint32_t)z0 | ((uint32_t)x1 << 16),
                            (uint32_t)y1 | ((uint32_t)z1 << 16), ((mask[b >> 5] >> (b & 31)) & 1u));
    }
}

enum : int { G_K = 0, G_LFX = 1, G_TIDX = 2, G_ECOUNT = 3, G_ELUCY = 4, G_TCOUNT = 5, G_TLUCY = 6, G_THYBRID = 7 };

__device__ __forceinline__ double T_of_x(const double *J, const double *Tg, int nT, double x)
{
    if (!(x > 0.0)) return 0.0;
    if (x <= J[0]) return Tg[0];
    if (x >= J[nT - 1]) return Tg[nT - 1];
    int lo = 0, hi = nT - 1;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (J[mid] <= x) lo = mid; else hi = mid;
    }
    const double f = log(x / J[lo]) / log(J[hi] / J[lo]);
    return Tg[lo] * exp(f * log(Tg[hi] / Tg[lo]));
}

// gathers one output array in canonical order (O12: E_count = k xi, E_lucy = xi L / 2^FX, T by inverting Eq. 4)
__global__ void k_gather(int what, void *__restrict__ out, const unsigned long long *__restrict__ cellw,
                         const unsigned long long *__restrict__ kcnt, const long long *__restrict__ lfx,
                         const double *__restrict__ J, const double *__restrict__ Tg, int nT, int nx, int ny, int nz,
                         int px, int pxy, double xi, double inv_fx, double cellfac, uint32_t tmask,
                         const int *__restrict__ mx_mat, const double *__restrict__ mx_frac, int comp,
                         const uint16_t *__restrict__ tidx1, const double *__restrict__ kmax_diag)
{
    // (mixtures, NEXT-3: kcnt / lfx are those of component `comp`, whose material and mass fraction enter Eq. 4)
    const size_t nc = (size_t)nx * ny * nz;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nc; i += (size_t)gridDim.x * blockDim.x) {
        const int ix = (int)(i % nx), iy = (int)((i / nx) % ny), iz = (int)(i / ((size_t)nx * ny));
        const size_t b = lin_index(ix, iy, iz, px, pxy), bs = (size_t)kCS * b;
        switch (what) {
        case G_K: reinterpret_cast<unsigned long long *>(out)[i] = kcnt[b]; break;
        case G_LFX: reinterpret_cast<long long *>(out)[i] = lfx[bs]; break;
        case G_TIDX:    // (a marker word -- the cube is divided into sub-cubes -- has no temperature index)
            reinterpret_cast<uint16_t *>(out)[i] = comp ? tidx1[b] : (cw_dusty(cellw[bs]) ? (uint16_t)cw_tidx(cellw[bs], tmask) : (uint16_t)0);
            break;
        case G_ECOUNT: reinterpret_cast<double *>(out)[i] = (double)kcnt[b] * xi; break;
        case G_ELUCY: reinterpret_cast<double *>(out)[i] = (double)lfx[bs] * inv_fx * xi; break;
        default: {
            const unsigned long long cw = cellw[bs];
            const double rho_c = cw_rho(cw);
            float T = 0.0f;
            if (cw_dusty(cw)) {
                double e = (what == G_TLUCY) ? (double)lfx[bs] * inv_fx : (double)kcnt[b];
                // Sect. 3.1 (reading Q39): the Eq. 9 energy below the threshold, the count above
                if (what == G_THYBRID) e = (rho_c * kmax_diag[cw_species(cw)] < kThinTau) ? (double)lfx[bs] * inv_fx : (double)kcnt[b];
                if (!mx_mat) T = (float)T_of_x(J + cw_species(cw) * nT, Tg, nT, e * cellfac / rho_c);
                else {
                    const int m = mx_mat[2 * cw_species(cw) + comp];
                    if (m >= 0) T = (float)T_of_x(J + m * nT, Tg, nT, e * cellfac / (rho_c * mx_frac[2 * cw_species(cw) + comp]));
                }
            }
            reinterpret_cast<float *>(out)[i] = T;
        }
        }
    }
}

__global__ void k_gather_sub(int what, void *__restrict__ out, const unsigned long long *__restrict__ cellw,
                             const unsigned long long *__restrict__ kcnt, const long long *__restrict__ lfx,
                             const double *__restrict__ J, const double *__restrict__ Tg, int nT, size_t off, size_t n, double xi,
                             double inv_fx, double cellfac, uint32_t tmask)
{
    // sub-cubes off .. off + n - 1 to out[0 .. n - 1]
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        const size_t i = off + o, bs = (size_t)kCS * i;
        switch (what) {
        case G_K: reinterpret_cast<unsigned long long *>(out)[o] = kcnt[i]; break;
        case G_LFX: reinterpret_cast<long long *>(out)[o] = lfx[bs]; break;
        case G_TIDX: reinterpret_cast<uint16_t *>(out)[o] = (uint16_t)cw_tidx(cellw[bs], tmask); break;
        case G_ECOUNT: reinterpret_cast<double *>(out)[o] = (double)kcnt[i] * xi; break;
        case G_ELUCY: reinterpret_cast<double *>(out)[o] = (double)lfx[bs] * inv_fx * xi; break;
        default: {
            const unsigned long long cw = cellw[bs];
            float T = 0.0f;
            if (cw_dusty(cw)) {
                const double e = (what == G_TLUCY) ? (double)lfx[bs] * inv_fx : (double)kcnt[i];
                T = (float)T_of_x(J + cw_species(cw) * nT, Tg, nT, e * cellfac / cw_rho(cw));
            }
            reinterpret_cast<float *>(out)[o] = T;
        }
        }
    }
}

// SED = counts xi / (dnu_j dOmega_bin), dOmega = 4 pi d|mu| (reading Q22)
__global__ void k_sed(double *__restrict__ out, const unsigned long long *__restrict__ sed, const double *__restrict__ dnu,
                      const double *__restrict__ mu, int ndir, int nf, double xi)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ndir * nf) {
        const int b = i / nf, j = i % nf;
        const double dom = kFourPi * (mu[b + 1] - mu[b]);
        out[i] = (double)sed[i] * xi / (dnu[j] * dom);
    }
}

// numbers the hot cells in bits 24-28 of their cell words (id 0 clears)
__global__ void k_set_hot(unsigned long long *__restrict__ cellw, const uint32_t *__restrict__ idx, const uint32_t *__restrict__ id, int n,
                          uint32_t shift, uint32_t mask)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        uint32_t *lo = reinterpret_cast<uint32_t *>(cellw + (size_t)kCS * idx[i]);
        *lo = (*lo & ~(mask << shift)) | (id[i] << shift);
    }
}

// cell words of a list of cells (the candidates for hot cells)
__global__ void k_fetch_words(const unsigned long long *__restrict__ cellw, const uint32_t *__restrict__ idx, unsigned long long *__restrict__ out, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = cellw[(size_t)kCS * idx[i]];
}

// ------------------------------------------------------------------------------------------------
// NEXT-2  ray tracer (Eq. 11-17)
// ------------------------------------------------------------------------------------------------
__host__ __device__ double planck_nu(double nu, double T);   // (defined with the host-side tables below)

__device__ __forceinline__ double phase_hg(double g, double cb)
{
    const double d = 1.0 + g * g - 2.0 * g * cb;
    return (1.0 - g * g) / (kFourPi * d * sqrt(d));        // Eq. 15, per steradian
}

// per-cell sum over the stored events of frequency slot `slot` of P_HG(beta) (the sum over beta of Eq. 16)
__global__ void k_sca_source(const mcrt_scatter_event *__restrict__ ev, unsigned long long n, int slot, double ezx, double ezy, double ezz,
                             const unsigned long long *__restrict__ cellw, const double *__restrict__ g, int nf, int j, int nx, int ny,
                             int px, int pxy, double *__restrict__ src)
{
    for (unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (unsigned long long)gridDim.x * blockDim.x) {
        const mcrt_scatter_event v = ev[e];
        if ((int)v.slot != slot) continue;
        const double qx = v.q[0], qy = v.q[1], qz = v.q[2];
        const double qn = sqrt(qx * qx + qy * qy + qz * qz);
        const double cb = (qx * ezx + qy * ezy + qz * ezz) / qn;
        const int ix = (int)(v.cell % (uint32_t)nx), iy = (int)((v.cell / (uint32_t)nx) % (uint32_t)ny), iz = (int)(v.cell / ((uint32_t)nx * (uint32_t)ny));
        const unsigned long long cw = cellw[(size_t)kCS * lin_index(ix, iy, iz, px, pxy)];
        atomicAdd(&src[v.cell], phase_hg(g[cw_species(cw) * nf + j], cb));
    }
}

struct RayParams {
    double ez[3], ex[3], ey[3];
    int inx, iny;
    double pix_cells, apix_d2, h, xi, inv_fx, cellfac, nu, inv_dnu;
    int nx, ny, nz, px, pxy, nT, from_lucy, j, nf;
};

__global__ void __launch_bounds__(128) k_ray_trace(RayParams R, const unsigned long long *__restrict__ cellw, const unsigned long long *__restrict__ kcnt,
                                                   const long long *__restrict__ lfx, const double *__restrict__ J, const double *__restrict__ Tg,
                                                   const double *__restrict__ kabs_j /*[ns] at this frequency*/, const double *__restrict__ src,
                                                   double *__restrict__ Fe, double *__restrict__ Fs)
{
    const int pixi = blockIdx.x * blockDim.x + threadIdx.x;
    if (pixi >= R.inx * R.iny) return;
    const int a = pixi % R.inx, b = pixi / R.inx;
    const int n[3] = {R.nx, R.ny, R.nz};
    const double u[3] = {-R.ez[0], -R.ez[1], -R.ez[2]};     // the walk runs from the observer's side inwards
    const double xa = ((double)a + 0.5 - 0.5 * R.inx) * R.pix_cells, yb = ((double)b + 0.5 - 0.5 * R.iny) * R.pix_cells;
    double r0[3], smin = -CUDART_INF, smax = CUDART_INF;
    bool miss = false;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        r0[q] = 0.5 * n[q] + xa * R.ex[q] + yb * R.ey[q];
        if (u[q] == 0.0) { if (!(r0[q] > 0.0 && r0[q] < (double)n[q])) miss = true; continue; }
        const double s1 = (0.0 - r0[q]) / u[q], s2 = ((double)n[q] - r0[q]) / u[q];
        smin = fmax(smin, fmin(s1, s2));
        smax = fmin(smax, fmax(s1, s2));
    }
    double fe = 0.0, fs = 0.0;
    if (!miss && smax > smin) {
        double p[3];
        int c[3], st[3];
        double iv[3], tm[3];
        bool inside = true;
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            p[q] = fmin(fmax(r0[q] + smin * u[q], 0.0), (double)n[q]);
            const double f = floor(p[q]);
            c[q] = (p[q] != f) ? (int)f : ((u[q] >= 0.0) ? (int)f : (int)f - 1);   // start cell (reading Q9)
            inside = inside && c[q] >= 0 && c[q] < n[q];
            st[q] = (u[q] > 0.0) ? 1 : ((u[q] < 0.0) ? -1 : 0);
            iv[q] = st[q] ? 1.0 / u[q] : CUDART_INF;
        }
        if (inside) {
#pragma unroll
            for (int q = 0; q < 3; ++q) tm[q] = mcrt::face_t(c[q], st[q], p[q], iv[q]);
            const double V = R.h * R.h * R.h;
            double t = 0.0, tau = 0.0;
            for (;;) {
                const int ax = (tm[0] <= tm[1] && tm[0] <= tm[2]) ? 0 : ((tm[1] <= tm[2]) ? 1 : 2);
                const double tn = tm[ax], l = (tn - t) * R.h;
                const unsigned long long cw = cellw[(size_t)kCS * lin_index(c[0], c[1], c[2], R.px, R.pxy)];
                if (cw_dusty(cw)) {
                    const size_t li = lin_index(c[0], c[1], c[2], R.px, R.pxy);
                    const size_t ci = ((size_t)c[2] * R.ny + c[1]) * R.nx + c[0];
                    const double rho_c = cw_rho(cw);
                    const int sp = cw_species(cw);
                    const double tc = kabs_j[sp] * rho_c * l;
                    const double e = R.from_lucy ? (double)lfx[(size_t)kCS * li] * R.inv_fx : (double)kcnt[li];
                    const double T = T_of_x(J + sp * R.nT, Tg, R.nT, e * R.cellfac / rho_c);
                    const double att = exp(-tau);
                    if (T > 0.0) fe += -expm1(-tc) * planck_nu(R.nu, T) * att;
                    fs += l / V * src[ci] * R.xi * R.inv_dnu * att;
                    tau += tc;
                }
                t = tn;
                c[ax] += st[ax];
                tm[ax] = mcrt::face_t(c[ax], st[ax], p[ax], iv[ax]);
                if (c[ax] < 0 || c[ax] >= n[ax]) break;
            }
        }
    }
    Fe[pixi] = fe * R.apix_d2;
    if (Fs) Fs[pixi] = fs * R.apix_d2;
}

// read-bandwidth probe: `passes` sweeps over a buffer, every thread summing 16-byte words with a grid stride, eight
// loads in flight
__global__ void __launch_bounds__(512) k_read_probe(const uint4 *__restrict__ buf, size_t n16, int passes, unsigned long long *__restrict__ sink)
{
    unsigned long long acc = 0ull;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int pass = 0; pass < passes; ++pass) {
        size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; i + 7 * stride < n16; i += 8 * stride) {
            uint4 v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = __ldcg(buf + i + k * stride);   // L2, not L1: what a resident grid's arrays see
#pragma unroll
            for (int k = 0; k < 8; ++k) acc += (unsigned long long)(v[k].x ^ v[k].y) + (unsigned long long)(v[k].z ^ v[k].w);
        }
        for (; i < n16; i += stride) { const uint4 v = __ldcg(buf + i); acc += (unsigned long long)(v.x ^ v.y) + (unsigned long long)(v.z ^ v.w); }
    }
    if (acc == 0x123456789abcdefull) sink[0] = acc;   // keeps the loads alive
}

__global__ void k_traj_math_test(const double *__restrict__ z, double *__restrict__ out, unsigned long long n)
{
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        double s, c;
        traj_sincos_turns(z[i], s, c);
        out[3 * i] = traj_log(z[i]); out[3 * i + 1] = s; out[3 * i + 2] = c;
    }
}

// The allocation-free variant of k_traj_math_test (mcrt_traj_math_device_static): its scratch -- the device copy of the
// input and the three output arrays -- lives in a file-scope device array of fixed size, 4 x 65536 doubles = 2 MiB,
// which every GPU that loads the library holds until the process exits.  All calls share it.
constexpr uint64_t kStaticMaxN = 65536;
constexpr int kStaticMaxDevices = 64;
static __device__ __align__(256) double g_static_scratch[4 * kStaticMaxN];
static std::atomic<double *> g_static_scratch_ptr[kStaticMaxDevices];   // its device address, per device ordinal (0 = not asked yet)

__global__ void k_traj_math_static(const double *__restrict__ z, double *__restrict__ ln_z, double *__restrict__ sn,
                                   double *__restrict__ cs, unsigned long long n)
{
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        double s, c;
        traj_sincos_turns(z[i], s, c);
        ln_z[i] = traj_log(z[i]); sn[i] = s; cs[i] = c;
    }
}

__global__ void k_philox_test(const uint32_t *__restrict__ ctr, const uint32_t *__restrict__ key, uint32_t *__restrict__ out,
                              unsigned long long n)
{
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        uint32_t o0, o1, o2, o3;
        philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1], o0, o1, o2, o3);
        out[4 * i] = o0; out[4 * i + 1] = o1; out[4 * i + 2] = o2; out[4 * i + 3] = o3;
    }
}

// ------------------------------------------------------------------------------------------------
// host-side tables (O1) -- small, built once per context
// ------------------------------------------------------------------------------------------------
__host__ __device__ double planck_nu(double nu, double T)
{
    const double x = kPlanckH * nu / (kBoltzK * T);
    return 2.0 * kPlanckH * nu * nu * nu / (kLightC * kLightC) / expm1(x);
}

double dplanck_nu_dT(double nu, double T)
{
    const double x = kPlanckH * nu / (kBoltzK * T);
    const double em = exp(-x);
    const double om = -expm1(-x);
    return 2.0 * kPlanckH * kPlanckH * nu * nu * nu * nu / (kLightC * kLightC * kBoltzK * T * T) * em / (om * om);
}

double make_cdf(const std::vector<double> &w, double *cdf)
{
    const size_t n = w.size();
    double tot = 0.0;
    for (size_t i = 0; i < n; ++i) tot += w[i];
    double acc = 0.0;
    for (size_t i = 0; i < n; ++i) {
        acc += w[i];
        cdf[i] = tot > 0.0 ? acc / tot : 0.0;
    }
    cdf[n - 1] = 1.0;
    return tot;
}

int fx_bits_for(uint64_t n)
{
    int cl = 0;
    while (((uint64_t)1 << cl) < n && cl < 63) ++cl;
    int fx = 58 - cl;
    if (fx > 40) fx = 40;
    if (fx < 0) fx = 0;
    return fx;
}

// Shared memory of a transport CTA is kept within the 196 KB carve-out: above it 28 KB of L1 remain for the walk's
// scattered loads, which measured 2x slower.

size_t transport_smem_bytes(int ns, int nf, int ndir, int mask0_words, int threads, bool record, int n_hot)
{
    return (size_t)(n_hot > 0 ? hot_smem_words(n_hot) : 0) * sizeof(unsigned int) +
           (size_t)(threads / 32) * pool_bytes_per_warp(record) + (size_t)(4 * ns * nf + nf + ndir + 1) * sizeof(double) +
           (size_t)(threads / 32) * 8 * sizeof(unsigned long long) + (size_t)2 * ndir * nf * sizeof(unsigned int) +
           (size_t)(MCRT_SMEM_MASK ? ((mask0_words + 1) & ~1) : 0) * sizeof(uint32_t) +
           (size_t)(nf < kPermSmem ? ((nf + 1 + 7) & ~7) : 0) * sizeof(unsigned short);
}

// The SM splits 256 KB between shared memory and L1 in fixed steps; a CTA also pays for the kernel's static shared
// memory and 1 KB the system reserves.  The walk's scattered loads live on what is left for L1: on torus256 the step
// from 164 KB to 196 KB of shared memory (92 -> 60 KB of L1) costs 5-6 % of the throughput (profiles/
// r02_experiments.md, section 5), so the hot-cell tallies only take what the carve-out the pools need leaves over.
constexpr size_t kSmemOverhead = 1024 + 64;
constexpr size_t kMaxTransportSmem = 196 * 1024 - kSmemOverhead;
size_t smem_carveout(size_t dynamic_bytes)
{
    static const int kb[] = {8, 16, 32, 64, 100, 132, 164, 196, 228};
    for (int k : kb)
        if (dynamic_bytes + kSmemOverhead <= (size_t)k * 1024) return (size_t)k * 1024;
    return (size_t)228 * 1024;
}

// Geometry of the three vacuum-mask levels: level-0 boxes of (1 << msh)^3 cells, msh >= 2 the smallest for
// which level 0 fits 32 KB of shared memory; each further level is 4x coarser per axis.
struct MaskGeom {
    int msh, nbx, nby, nbz, mwords;
};

MaskGeom mask_geom(int nx, int ny, int nz)
{
    MaskGeom g;
    g.msh = 2;
    for (;;) {
        const size_t e = (size_t)1 << g.msh;
        const size_t bits = ((nx + e - 1) / e) * ((ny + e - 1) / e) * ((nz + e - 1) / e);
        if (bits <= ((size_t)1 << 18)) break;
        ++g.msh;
    }
    const int e = 1 << g.msh;
    g.nbx = (nx + e - 1) / e; g.nby = (ny + e - 1) / e; g.nbz = (nz + e - 1) / e;
    g.mwords = (g.nbx * g.nby * g.nbz + 31) / 32;
    return g;
}

int stream_grid(size_t n)
{
    size_t b = (n + 255) / 256;
    if (b > 148 * 16) b = 148 * 16;
    if (b < 1) b = 1;
    return (int)b;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------------
extern "C" {

const char *mcrt_version(void) { return MCRT_VERSION_STRING; }

const char *mcrt_last_error(const mcrt_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

void mcrt_default_opts(mcrt_run_opts *o)
{
    if (!o) return;
    memset(o, 0, sizeof(*o));
    o->mode = MCRT_MODE_BW_EPOCH;
    o->sweep_T_from_lucy = 1;
    o->reset_tallies = 1;
    o->epoch_growth = 2.0;
    o->part_count = 1;
}

int mcrt_workspace_bytes(int nx, int ny, int nz, int n_species, int n_nu, int n_T, int n_dir, uint64_t n_digests,
                         size_t *bytes_out)
{
    if (!bytes_out || nx < 1 || ny < 1 || nz < 1 || n_species < 1 || n_nu < 2 || n_T < 2 || n_dir < 1) return MCRT_EINVAL;
    const MaskGeom mg = mask_geom(nx, ny, nz);
    const size_t nbricks = (size_t)mg.nbx * mg.nby * mg.nbz;
    const size_t ncp = (size_t)((nx + 2 * kGuard + MCRT_PITCH_ALIGN - 1) / MCRT_PITCH_ALIGN * MCRT_PITCH_ALIGN) * (ny + 2 * kGuard) * (nz + 2 * kGuard);
    size_t b = 0;
    auto add = [&b](size_t v) { b += align_up(v ? v : 1, 256); };
    add((ncp + 1) * sizeof(uint2) * kCS);   // cell words (kCS = 2: 16-byte records of cell word + Lucy tally)
    add((size_t)mg.mwords * 4);          // vacuum mask
    add(nbricks * sizeof(uint4));        // empty boxes of the J phase
    add((size_t)(mg.nbx + 1) * (mg.nby + 1) * (mg.nbz + 1) * sizeof(int));   // summed-area scratch
    if (kCS == 1) add(ncp * sizeof(long long));   // Lucy tally
    add(ncp * sizeof(long long));        // k
    add(ncp * sizeof(long long));        // k_prev
    add(ncp * 8);                        // scratch (staging of inputs / outputs / exchanged tallies)
    add(CNT_N * 8 + 64);                 // counters (+ validation flags)
    const size_t nsf = (size_t)n_species * n_nu;
    for (int i = 0; i < 4; ++i) add(nsf * 8);
    add((size_t)n_nu * 8); add((size_t)n_nu * 8);            // srccdf, dnu
    add((size_t)n_species * n_T * 8); add((size_t)n_T * 8);  // J, Tg
    { const size_t nfs = (size_t)(n_nu + 1 + 15) / 16 * 16; add((size_t)n_species * n_T * nfs * 8); add((size_t)n_species * n_T * nfs * 8); }   // cdf_B, cdf_dB (Eytzinger rows)
    add((size_t)(n_nu + 1) * 2);                             // their permutation
    add((size_t)(n_dir + 1) * 8);
    add((size_t)n_dir * n_nu * 8); add((size_t)n_dir * n_nu * 8);
    add((size_t)n_dir * n_nu * 8);                           // SED staging
    add((size_t)(5 * (kHot + 1) + 4 * 1400) * sizeof(uint32_t));   // hot-cell table and staging (mcrt_source)
    if (n_digests) add(n_digests * sizeof(mcrt_digest));
    *bytes_out = b + 4096;
    return MCRT_OK;
}

int mcrt_grid_create(mcrt_ctx **out, int nx, int ny, int nz, double cell_size_cm, const float *rho, const uint8_t *species,
                     int n_species, mcrt_mem where, void *workspace, size_t workspace_bytes)
{
    if (!out) return fail(nullptr, MCRT_EINVAL, "out is NULL");
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1) return fail(nullptr, MCRT_EINVAL, "nx, ny, nz must be >= 1");
    if (nx > 2040 || ny > 2040 || nz > 1016) return fail(nullptr, MCRT_EINVAL, "grid too large: nx, ny <= 2040 and nz <= 1016");
    if ((size_t)(nx + 2 * kGuard) * (ny + 2 * kGuard) * (nz + 2 * kGuard) > ((size_t)1 << 30)) return fail(nullptr, MCRT_EINVAL, "grid larger than 2^30 cells (guard shell included)");
    if (!(cell_size_cm > 0.0) || !isfinite(cell_size_cm)) return fail(nullptr, MCRT_EINVAL, "cell_size_cm must be > 0");
    if (!rho || !species) return fail(nullptr, MCRT_EINVAL, "rho / species is NULL");
    if (n_species < 1 || n_species > 255) return fail(nullptr, MCRT_EINVAL, "n_species must be in 1..255");
    if (workspace && ((uintptr_t)workspace & 255u)) return fail(nullptr, MCRT_EINVAL, "workspace must be 256-byte aligned");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1)
        return fail(nullptr, MCRT_ECUDA, "no CUDA device: this library has no CPU fallback");
    mcrt_ctx *c = new mcrt_ctx();
    cudaGetDevice(&c->device);
    c->nx = nx; c->ny = ny; c->nz = nz; c->ns = n_species; c->h = cell_size_cm;
    {
        const MaskGeom g = mask_geom(nx, ny, nz);
        c->msh = g.msh; c->mwords = g.mwords;
        c->nbx = g.nbx; c->nby = g.nby; c->nbz = g.nbz;
    }
    c->nc = (size_t)nx * ny * nz;
    c->px = (nx + 2 * kGuard + MCRT_PITCH_ALIGN - 1) / MCRT_PITCH_ALIGN * MCRT_PITCH_ALIGN; c->pxy = c->px * (ny + 2 * kGuard);
    c->ncp = (size_t)c->pxy * (nz + 2 * kGuard);
    c->ws = (char *)workspace; c->ws_bytes = workspace_bytes; c->ws_owned_by_caller = workspace != nullptr;
    int rc;
#define GC_TRY(expr)                                                       \
    do {                                                                   \
        rc = (expr);                                                       \
        if (rc != MCRT_OK) { g_create_error = c->err; mcrt_destroy(c); return rc; } \
    } while (0)
#define GC_CUDA(expr)                                                                                  \
    do {                                                                                               \
        cudaError_t e__ = (expr);                                                                      \
        if (e__ != cudaSuccess) {                                                                      \
            g_create_error = std::string(#expr) + ": " + cudaGetErrorString(e__);                      \
            mcrt_destroy(c);                                                                           \
            return MCRT_ECUDA;                                                                         \
        }                                                                                              \
    } while (0)
    GC_TRY(ws_alloc(c, (void **)&c->cellw, (c->ncp + 1) * sizeof(uint2) * kCS));
    GC_TRY(ws_alloc(c, (void **)&c->vmask, (size_t)c->mwords * 4));
    GC_TRY(ws_alloc(c, (void **)&c->vbox, (size_t)c->nbx * c->nby * c->nbz * sizeof(uint4)));
    GC_TRY(ws_alloc(c, (void **)&c->vsat, (size_t)(c->nbx + 1) * (c->nby + 1) * (c->nbz + 1) * sizeof(int)));
    if (kCS == 1) GC_TRY(ws_alloc(c, (void **)&c->lfx, c->ncp * sizeof(long long)));
    else c->lfx = reinterpret_cast<long long *>(c->cellw + 1);   // second word of every 16-byte cell record
    GC_TRY(ws_alloc(c, (void **)&c->kabs_cnt, c->ncp * sizeof(long long)));
    GC_TRY(ws_alloc(c, (void **)&c->kprev, c->ncp * sizeof(long long)));
    GC_TRY(ws_alloc(c, (void **)&c->scratch, c->ncp * 8));   // staging: inputs, outputs, the Lucy tallies of an exchange
    GC_TRY(ws_alloc(c, (void **)&c->counters, CNT_N * 8 + 64));
    GC_CUDA(cudaMemsetAsync(c->counters, 0, CNT_N * 8 + 64, c->stream));
    const float *d_rho = rho;
    const uint8_t *d_sp = species;
    if (where == MCRT_HOST) {
        float *sr = (float *)c->scratch;
        uint8_t *ss = (uint8_t *)c->scratch + c->nc * 4;
        GC_CUDA(cudaMemcpyAsync(sr, rho, c->nc * 4, cudaMemcpyHostToDevice, c->stream));
        GC_CUDA(cudaMemcpyAsync(ss, species, c->nc, cudaMemcpyHostToDevice, c->stream));
        d_rho = sr; d_sp = ss;
    }
    unsigned long long *bad = c->counters + CNT_N;
    k_pack_grid<<<stream_grid(c->ncp), 256, 0, c->stream>>>(d_rho, d_sp, c->cellw, nx, ny, nz, c->px, c->pxy, c->ncp, n_species, bad);
    GC_CUDA(cudaGetLastError());
    GC_CUDA(cudaMemsetAsync(c->vmask, 0, (size_t)c->mwords * 4, c->stream));
    {
        const size_t nbr = (size_t)c->nbx * c->nby * c->nbz;
        k_build_mask0<<<stream_grid(nbr), 256, 0, c->stream>>>(c->cellw, c->vmask, nx, ny, nz, c->px, c->pxy, c->msh, c->nbx,
                                                             c->nby, c->nbz);
        if (MCRT_VAC_SPECIES) k_vac_species<<<stream_grid(c->nc), 256, 0, c->stream>>>(c->cellw, nx, ny, nz, c->px, c->pxy);
        GC_CUDA(cudaMemsetAsync(c->vsat, 0, (size_t)(c->nbx + 1) * (c->nby + 1) * (c->nbz + 1) * sizeof(int), c->stream));
        k_sat_pass<<<stream_grid((size_t)c->nby * c->nbz), 256, 0, c->stream>>>(c->vmask, c->vsat, c->nbx, c->nby, c->nbz, 0);
        k_sat_pass<<<stream_grid((size_t)c->nbx * c->nbz), 256, 0, c->stream>>>(c->vmask, c->vsat, c->nbx, c->nby, c->nbz, 1);
        k_sat_pass<<<stream_grid((size_t)c->nbx * c->nby), 256, 0, c->stream>>>(c->vmask, c->vsat, c->nbx, c->nby, c->nbz, 2);
        k_grow_boxes<<<stream_grid(nbr), 256, 0, c->stream>>>(c->vmask, c->vsat, c->vbox, c->nbx, c->nby, c->nbz);
    }
    GC_CUDA(cudaGetLastError());
    GC_CUDA(cudaMemset2DAsync(c->lfx, 8 * kCS, 0, 8, c->ncp, c->stream));
    GC_CUDA(cudaMemsetAsync(c->kabs_cnt, 0, c->ncp * 8, c->stream));
    GC_CUDA(cudaMemsetAsync(c->kprev, 0, c->ncp * 8, c->stream));
    unsigned long long hbad[3] = {0, 0, 0};
    GC_CUDA(cudaMemcpyAsync(hbad, bad, 24, cudaMemcpyDeviceToHost, c->stream));
    GC_CUDA(cudaStreamSynchronize(c->stream));
    if (hbad[0] || hbad[1]) {
        g_create_error = hbad[0] ? "rho holds negative, NaN or infinite values" : "species index >= n_species";
        mcrt_destroy(c);
        return MCRT_EINVAL;
    }
    c->n_dusty = hbad[2];
    {
        int l2 = 0;
        if (cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, c->device) == cudaSuccess && l2 > 0) c->l2_bytes = (size_t)l2;
    }
#undef GC_TRY
#undef GC_CUDA
    *out = c;
    return MCRT_OK;
}

int mcrt_set_stream(mcrt_ctx *c, void *cuda_stream)
{
    if (!c) return MCRT_EINVAL;
    c->stream = (cudaStream_t)cuda_stream;
    return MCRT_OK;
}

int mcrt_dust_tables(mcrt_ctx *c, int n_nu, const double *nu_hz, const double *kappa_abs, const double *kappa_sca,
                     const double *g, int n_T, const double *T_grid)
{
    if (!c) return MCRT_EINVAL;
    if (c->have_tables) return fail(c, MCRT_ESTATE, "mcrt_dust_tables may be called once per context");
    if (!nu_hz || !kappa_abs || !kappa_sca || !g || !T_grid) return fail(c, MCRT_EINVAL, "NULL table pointer");
    if (n_nu < 2 || n_nu > 65535 || n_T < 2 || n_T > 65535) return fail(c, MCRT_EINVAL, "n_nu and n_T must be in 2..65535");
    for (int j = 0; j < n_nu; ++j) {
        if (!(nu_hz[j] > 0.0) || !isfinite(nu_hz[j]) || (j && !(nu_hz[j] > nu_hz[j - 1])))
            return fail(c, MCRT_EINVAL, "nu_hz must be positive and strictly ascending");
    }
    for (int m = 0; m < n_T; ++m)
        if (!(T_grid[m] > 0.0) || !isfinite(T_grid[m]) || (m && !(T_grid[m] > T_grid[m - 1])))
            return fail(c, MCRT_EINVAL, "T_grid must be positive and strictly ascending");
    const int ns = c->ns;
    const size_t nsf = (size_t)ns * n_nu;
    for (size_t i = 0; i < nsf; ++i) {
        if (!(kappa_abs[i] >= 0.0) || !(kappa_sca[i] >= 0.0) || !isfinite(kappa_abs[i]) || !isfinite(kappa_sca[i]))
            return fail(c, MCRT_EINVAL, "kappa must be finite and >= 0");
        if (!(kappa_abs[i] + kappa_sca[i] > 0.0)) return fail(c, MCRT_EINVAL, "kappa_abs + kappa_sca must be > 0");
        if (!(fabs(g[i]) < 1.0)) return fail(c, MCRT_EINVAL, "|g| must be < 1");
    }
    if (transport_smem_bytes(ns, n_nu, 16, c->mwords, 256, true, 0) > kMaxTransportSmem)
        return fail(c, MCRT_EINVAL, "n_species * n_nu too large for the shared-memory tables");
    c->nf = n_nu; c->nT = n_T;
    // low half of the cell word: species 0-7 | temperature index (12 or 16 bits) | hot-cell number (9 or 5 bits) | rho 29-31
    if (n_T <= 4096) { c->tidx_mask = 0xfffu; c->hot_shift = 20; c->hot_mask = 511u; c->hot_max = 511; }
    else { c->tidx_mask = 0xffffu; c->hot_shift = 24; c->hot_mask = 31u; c->hot_max = 31; }
    c->nu.assign(nu_hz, nu_hz + n_nu);
    c->kabs.assign(kappa_abs, kappa_abs + nsf);
    c->ksca.assign(kappa_sca, kappa_sca + nsf);
    c->g.assign(g, g + nsf);
    c->Tg.assign(T_grid, T_grid + n_T);
    // bin widths: edges at the geometric means of neighbours, end bins extrapolated with the neighbouring ratio
    c->dnu.resize(n_nu);
    {
        std::vector<double> edge(n_nu + 1);
        for (int j = 1; j < n_nu; ++j) edge[j] = sqrt(c->nu[j - 1] * c->nu[j]);
        edge[0] = c->nu[0] * sqrt(c->nu[0] / c->nu[1]);
        edge[n_nu] = c->nu[n_nu - 1] * sqrt(c->nu[n_nu - 1] / c->nu[n_nu - 2]);
        for (int j = 0; j < n_nu; ++j) c->dnu[j] = edge[j + 1] - edge[j];
    }
    c->kext_h.resize(nsf); c->kabs_h.resize(nsf); c->albedo.resize(nsf);
    for (size_t i = 0; i < nsf; ++i) {
        const double kext = c->kabs[i] + c->ksca[i];
        c->kext_h[i] = kext * c->h;        // optical depth per unit density per cell length (Eq. 2)
        c->kabs_h[i] = c->kabs[i] * c->h;
        c->albedo[i] = c->ksca[i] / kext;
    }
    c->J.resize((size_t)ns * n_T);
    c->cdfB.resize(nsf * n_T);
    c->cdfdB.resize(nsf * n_T);
    std::vector<double> w(n_nu);
    for (int s = 0; s < ns; ++s)
        for (int m = 0; m < n_T; ++m) {
            const size_t row = ((size_t)s * n_T + m) * n_nu;
            for (int j = 0; j < n_nu; ++j) w[j] = c->kabs[(size_t)s * n_nu + j] * planck_nu(c->nu[j], c->Tg[m]) * c->dnu[j];
            c->J[(size_t)s * n_T + m] = make_cdf(w, &c->cdfB[row]);      // Eq. 4 left side, Eq. 5
            for (int j = 0; j < n_nu; ++j) w[j] = c->kabs[(size_t)s * n_nu + j] * dplanck_nu_dT(c->nu[j], c->Tg[m]) * c->dnu[j];
            make_cdf(w, &c->cdfdB[row]);                                  // Eq. 10
        }
    int rc;
    if ((rc = ws_alloc(c, (void **)&c->d_kext_h, nsf * 8))) return rc;
    if ((rc = ws_alloc(c, (void **)&c->d_kabs_fx, nsf * 8))) return rc;
    if ((rc = ws_alloc(c, (void **)&c->d_albedo, nsf * 8))) return rc;
    if ((rc = ws_alloc(c, (void **)&c->d_g, nsf * 8))) return rc;
    if ((rc = ws_alloc(c, (void **)&c->d_srccdf, (size_t)n_nu * 8))) return rc;
    if ((rc = ws_alloc(c, (void **)&c->d_dnu, (size_t)n_nu * 8))) return rc;
    if ((rc = ws_alloc(c, (void **)&c->d_J, (size_t)ns * n_T * 8))) return rc;
    if ((rc = ws_alloc(c, (void **)&c->d_Tg, (size_t)n_T * 8))) return rc;
    // the re-emission rows go to the device in Eytzinger order (lower_bound_eytzinger), 1-based, rows padded to 16 doubles
    c->nfs = (n_nu + 1 + 15) / 16 * 16;
    c->perm.assign(n_nu + 1, 0);
    {
        int next = 0;
        std::vector<int> stack;               // in-order walk of the implicit tree: node k gets the next ascending position
        int k = 1;
        while (!stack.empty() || k <= n_nu) {
            while (k <= n_nu) { stack.push_back(k); k = 2 * k; }
            k = stack.back(); stack.pop_back();
            c->perm[k] = (unsigned short)next++;
            k = 2 * k + 1;
        }
    }
    const size_t rows = (size_t)ns * n_T;
    std::vector<double> eyt(rows * c->nfs, 2.0);   // (padding above every CDF value: never taken)
    if ((rc = ws_alloc(c, (void **)&c->d_cdfB, rows * c->nfs * 8))) return rc;
    if ((rc = ws_alloc(c, (void **)&c->d_cdfdB, rows * c->nfs * 8))) return rc;
    if ((rc = ws_alloc(c, (void **)&c->d_perm, (size_t)(n_nu + 1) * 2))) return rc;
    CUDA_TRY(c, cudaMemcpyAsync(c->d_kext_h, c->kext_h.data(), nsf * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_albedo, c->albedo.data(), nsf * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_g, c->g.data(), nsf * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_dnu, c->dnu.data(), (size_t)n_nu * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_J, c->J.data(), (size_t)ns * n_T * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_Tg, c->Tg.data(), (size_t)n_T * 8, cudaMemcpyHostToDevice, c->stream));
    for (int pass = 0; pass < 2; ++pass) {
        const std::vector<double> &src = pass ? c->cdfdB : c->cdfB;
        for (size_t r = 0; r < rows; ++r)
            for (int k = 1; k <= n_nu; ++k) eyt[r * c->nfs + k] = src[r * n_nu + c->perm[k]];
        CUDA_TRY(c, cudaMemcpyAsync(pass ? c->d_cdfdB : c->d_cdfB, eyt.data(), rows * c->nfs * 8, cudaMemcpyHostToDevice, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    }
    CUDA_TRY(c, cudaMemcpyAsync(c->d_perm, c->perm.data(), (size_t)(n_nu + 1) * 2, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    c->have_tables = true;
    return MCRT_OK;
}

static int apply_hot(mcrt_ctx *c, int n_use);
static int check_overflow(mcrt_ctx *c);

int mcrt_subgrid(mcrt_ctx *c, int R, uint64_t n_sub, const int64_t *cube, const float *rho_sub, const uint8_t *species_sub)
{
    if (!c) return MCRT_EINVAL;
    if (c->subR) return fail(c, MCRT_ESTATE, "mcrt_subgrid may be called once per context");
    if (c->last_n || c->run.active) return fail(c, MCRT_ESTATE, "mcrt_subgrid after a run");
    if (c->mix) return fail(c, MCRT_EINVAL, "mcrt_subgrid is not available with dust mixtures");
    if (R != 2 && R != 4 && R != 8) return fail(c, MCRT_EINVAL, "R must be 2, 4 or 8");
    if (n_sub < 1 || n_sub > ((uint64_t)1 << 22) || !cube || !rho_sub || !species_sub) return fail(c, MCRT_EINVAL, "1 <= n_sub <= 2^22 divided cubes");
    const size_t R3 = (size_t)R * R * R, n = (size_t)n_sub * R3;
    {
        std::vector<int64_t> sorted(cube, cube + n_sub);
        std::sort(sorted.begin(), sorted.end());
        if (sorted.front() < 0 || (uint64_t)sorted.back() >= c->nc) return fail(c, MCRT_EINVAL, "cube index out of range");
        for (size_t i = 1; i < sorted.size(); ++i)
            if (sorted[i] == sorted[i - 1]) return fail(c, MCRT_EINVAL, "a cube is listed twice");
    }
    long long *d_cube = nullptr; float *d_rho = nullptr; uint8_t *d_sp = nullptr;
    bool ok = cudaMalloc((void **)&c->sub_cellw, n * kCS * 8) == cudaSuccess && cudaMalloc((void **)&c->sub_lfx, n * kCS * 8) == cudaSuccess &&
              cudaMalloc((void **)&c->sub_kcnt, n * 8) == cudaSuccess && cudaMalloc((void **)&c->sub_kprev, n * 8) == cudaSuccess &&
              cudaMalloc((void **)&d_cube, n_sub * 8) == cudaSuccess && cudaMalloc((void **)&d_rho, n * 4) == cudaSuccess &&
              cudaMalloc((void **)&d_sp, n) == cudaSuccess;
    int rc = MCRT_OK;
    unsigned long long bad[2] = {0ull, 0ull};
    unsigned long long *d_bad = c->counters + CNT_N;
    cudaError_t e = cudaSuccess;
    if (!ok) rc = fail(c, MCRT_ENOMEM, "cudaMalloc of the sub-cube arrays failed");
    if (!rc) {
        e = cudaMemcpyAsync(d_cube, cube, n_sub * 8, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_rho, rho_sub, n * 4, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_sp, species_sub, n, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(d_bad, 0, 16, c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->sub_lfx, 0, n * kCS * 8, c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->sub_kcnt, 0, n * 8, c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->sub_kprev, 0, n * 8, c->stream);
        if (e == cudaSuccess) {
            k_pack_sub<<<stream_grid(n), 256, 0, c->stream>>>(c->cellw, c->sub_cellw, d_cube, d_rho, d_sp, (size_t)n_sub, (int)R3, c->nx, c->ny,
                                                             c->nz, c->px, c->pxy, c->ns, d_bad);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(bad, d_bad, 16, cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) rc = fail(c, MCRT_ECUDA, cudaGetErrorString(e));
    }
    cudaFree(d_cube); cudaFree(d_rho); cudaFree(d_sp);
    if (!rc && bad[0]) rc = fail(c, MCRT_EINVAL, "a divided cube must have a density > 0 in the grid (a placeholder: its dust is in its sub-cubes)");
    if (!rc && bad[1]) rc = fail(c, MCRT_EINVAL, "sub-cube densities must be finite and >= 0, species < n_species");
    if (rc) return rc;      // (the context is unusable after a failure that has already rewritten cell words: destroy it)
    c->subR = R; c->sub_shift = R == 2 ? 1 : (R == 4 ? 2 : 3); c->n_sub = (size_t)n_sub; c->n_subcells = n;
    // no per-CTA copies of tallies on divided grids (a cell near the source may be a divided cube)
    if ((rc = apply_hot(c, 0))) return rc;
    c->hot_cand.clear();
    return MCRT_OK;
}

int mcrt_read_subcells(mcrt_ctx *c, double *E_abs_count, double *E_abs_lucy, float *T_count, float *T_lucy, uint64_t *k_abs,
                       int64_t *lucy_fx, uint16_t *tidx, mcrt_mem where)
{
    if (!c) return MCRT_EINVAL;
    if (!c->subR) return fail(c, MCRT_ESTATE, "mcrt_read_subcells without mcrt_subgrid");
    if (!c->last_n) return fail(c, MCRT_ESTATE, "mcrt_read_subcells before mcrt_run");
    if (c->run.active) return fail(c, MCRT_ESTATE, "mcrt_read_subcells inside mcrt_run_begin .. mcrt_run_end");
    int rc = check_overflow(c);
    if (rc) return rc;
    const double hs = c->h / (double)c->subR;
    const double cellfac = c->xi / (kFourPi * hs * hs * hs);
    struct { int what; void *dst; size_t elem; } outs[7] = {{G_ECOUNT, E_abs_count, 8}, {G_ELUCY, E_abs_lucy, 8}, {G_TCOUNT, T_count, 4},
                                                            {G_TLUCY, T_lucy, 4}, {G_K, k_abs, 8}, {G_LFX, lucy_fx, 8}, {G_TIDX, tidx, 2}};
    for (auto &o : outs) {
        if (!o.dst) continue;
        // host reads are staged through the context's scratch array (one value per grid cell), a piece at a time
        const size_t piece = (where == MCRT_DEVICE) ? c->n_subcells : std::min(c->n_subcells, c->nc);
        for (size_t off = 0; off < c->n_subcells; off += piece) {
            const size_t n = std::min(piece, c->n_subcells - off);
            void *dev = (where == MCRT_DEVICE) ? o.dst : c->scratch;
            k_gather_sub<<<stream_grid(n), 256, 0, c->stream>>>(o.what, dev, c->sub_cellw, c->sub_kcnt, c->sub_lfx, c->d_J, c->d_Tg, c->nT, off,
                                                               n, c->xi, ldexp(1.0, -c->fx), cellfac, c->tidx_mask);
            CUDA_TRY(c, cudaGetLastError());
            if (where == MCRT_HOST) {
                CUDA_TRY(c, cudaMemcpyAsync((char *)o.dst + off * o.elem, dev, n * o.elem, cudaMemcpyDeviceToHost, c->stream));
                CUDA_TRY(c, cudaStreamSynchronize(c->stream));
            }
        }
    }
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MCRT_OK;
}

int mcrt_dust_mixtures(mcrt_ctx *c, const int32_t *n_components, const int32_t *material, const double *fraction)
{
    if (!c) return MCRT_EINVAL;
    if (!c->have_tables) return fail(c, MCRT_ESTATE, "call mcrt_dust_tables before mcrt_dust_mixtures");
    if (c->mix) return fail(c, MCRT_ESTATE, "mcrt_dust_mixtures may be called once per context");
    if (c->last_n || c->run.active) return fail(c, MCRT_ESTATE, "mcrt_dust_mixtures after a run");
    if (!n_components || !material || !fraction) return fail(c, MCRT_EINVAL, "NULL mixture table");
    const int ns = c->ns, nf = c->nf;
    for (int x = 0; x < ns; ++x) {
        if (n_components[x] < 1 || n_components[x] > 2) return fail(c, MCRT_EINVAL, "a mixture has 1 or 2 components");
        double tot = 0.0;
        for (int k = 0; k < n_components[x]; ++k) {
            if (material[2 * x + k] < 0 || material[2 * x + k] >= ns) return fail(c, MCRT_EINVAL, "material index out of range");
            if (!(fraction[2 * x + k] > 0.0) || !isfinite(fraction[2 * x + k])) return fail(c, MCRT_EINVAL, "mass fractions must be > 0");
            tot += fraction[2 * x + k];
        }
        if (fabs(tot - 1.0) > 1e-12) return fail(c, MCRT_EINVAL, "the mass fractions of a mixture must add up to 1");
    }
    const size_t nsf = (size_t)ns * nf;
    c->mx_ncomp.assign(n_components, n_components + ns);
    c->mx_mat.assign(2 * (size_t)ns, -1);
    c->mx_frac.assign(2 * (size_t)ns, 0.0);
    c->mx_S0.assign(nsf, 0.0); c->mx_A0.assign(nsf, 1.0); c->kabs1_h.assign(nsf, 0.0);
    std::vector<double> thr(2 * nsf);
    // readings Q34 / Q35: extinction adds up in component order; the event uniform's thresholds
    for (int x = 0; x < ns; ++x) {
        for (int k = 0; k < n_components[x]; ++k) { c->mx_mat[2 * x + k] = material[2 * x + k]; c->mx_frac[2 * x + k] = fraction[2 * x + k]; }
        const int m0 = material[2 * x];
        for (int j = 0; j < nf; ++j) {
            const size_t i = (size_t)x * nf + j, i0 = (size_t)m0 * nf + j;
            if (n_components[x] == 1) {       // the material itself: the arithmetic of mcrt_dust_tables
                const double kext = c->kabs[i0] + c->ksca[i0];
                c->kext_h[i] = kext * c->h;
                c->kabs_h[i] = c->kabs[i0] * c->h;
                c->albedo[i] = c->ksca[i0] / kext;
                c->mx_S0[i] = c->albedo[i]; c->mx_A0[i] = 1.0;
            } else {
                const size_t i1 = (size_t)material[2 * x + 1] * nf + j;
                const double f0 = fraction[2 * x], f1 = fraction[2 * x + 1];
                const double ka0 = f0 * c->kabs[i0], ks0 = f0 * c->ksca[i0], ka1 = f1 * c->kabs[i1], ks1 = f1 * c->ksca[i1];
                const double kext = (ka0 + ks0) + (ka1 + ks1);
                c->kext_h[i] = kext * c->h;
                c->kabs_h[i] = ka0 * c->h;
                c->kabs1_h[i] = ka1 * c->h;
                c->mx_S0[i] = ks0 / kext;
                c->albedo[i] = (ks0 + ks1) / kext;
                c->mx_A0[i] = ((ks0 + ks1) + ka0) / kext;
            }
            thr[2 * i] = c->mx_S0[i]; thr[2 * i + 1] = c->mx_A0[i];
        }
    }
    // NB: c->kabs / c->ksca / c->g stay the MATERIALS' tables; kext_h, kabs_h and albedo are now the mixtures'
    const size_t cells = c->ncp * (size_t)kCS;
    if (cudaMalloc((void **)&c->d_mx_ncomp, ns * sizeof(int)) != cudaSuccess || cudaMalloc((void **)&c->d_mx_mat, 2 * ns * sizeof(int)) != cudaSuccess ||
        cudaMalloc((void **)&c->d_mx_frac, 2 * ns * 8) != cudaSuccess || cudaMalloc((void **)&c->d_mx_thr, 2 * nsf * 8) != cudaSuccess ||
        cudaMalloc((void **)&c->d_kabs1_fx, nsf * 8) != cudaSuccess || cudaMalloc((void **)&c->lfx1, cells * 8) != cudaSuccess ||
        cudaMalloc((void **)&c->kcnt1, c->ncp * 8) != cudaSuccess || cudaMalloc((void **)&c->kprev1, c->ncp * 8) != cudaSuccess ||
        cudaMalloc((void **)&c->tidx1, c->ncp * 2) != cudaSuccess)
        return fail(c, MCRT_ENOMEM, "cudaMalloc of the second component's arrays failed");
    CUDA_TRY(c, cudaMemcpyAsync(c->d_mx_ncomp, c->mx_ncomp.data(), ns * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_mx_mat, c->mx_mat.data(), 2 * ns * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_mx_frac, c->mx_frac.data(), 2 * ns * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_mx_thr, thr.data(), 2 * nsf * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_kext_h, c->kext_h.data(), nsf * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_albedo, c->albedo.data(), nsf * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->lfx1, 0, cells * 8, c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->kcnt1, 0, c->ncp * 8, c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->kprev1, 0, c->ncp * 8, c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->tidx1, 0, c->ncp * 2, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));   // thr and the host vectors must outlive the copies
    c->mix = true;
    return MCRT_OK;
}

// Number the first n_use candidates (nearest first) as hot cells 1..n_use in their cell words, after clearing the
// numbering in force.
static int apply_hot(mcrt_ctx *c, int n_use)
{
    if (n_use > (int)c->hot_cand.size()) n_use = (int)c->hot_cand.size();
    if (n_use == c->n_hot) return MCRT_OK;
    uint32_t *d_stage = c->d_hot_idx + (kHot + 1);
    std::vector<uint32_t> h_idx, h_id;
    for (int i = 1; i <= c->n_hot; ++i) { h_idx.push_back(c->hot_idx[i]); h_id.push_back(0u); }
    c->n_hot = n_use;
    c->hot_idx.assign(kHot + 1, 0u);
    for (int i = 1; i <= c->n_hot; ++i) { c->hot_idx[i] = c->hot_cand[i - 1]; h_idx.push_back(c->hot_idx[i]); h_id.push_back((uint32_t)i); }
    const int n = (int)h_idx.size();       // <= 2 kHot
    if (n) {
        CUDA_TRY(c, cudaMemcpyAsync(d_stage, h_idx.data(), n * 4, cudaMemcpyHostToDevice, c->stream));
        CUDA_TRY(c, cudaMemcpyAsync(d_stage + 2 * (kHot + 1), h_id.data(), n * 4, cudaMemcpyHostToDevice, c->stream));
        k_set_hot<<<(n + 127) / 128, 128, 0, c->stream>>>(c->cellw, d_stage, d_stage + 2 * (kHot + 1), n, c->hot_shift, c->hot_mask);
        CUDA_TRY(c, cudaGetLastError());
    }
    CUDA_TRY(c, cudaMemcpyAsync(c->d_hot_idx, c->hot_idx.data(), (kHot + 1) * 4, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MCRT_OK;
}

int mcrt_source(mcrt_ctx *c, double L_erg_s, double T_star_K, const double *L_nu_weights, const double pos_cm[3])
{
    if (!c) return MCRT_EINVAL;
    if (!c->have_tables) return fail(c, MCRT_ESTATE, "call mcrt_dust_tables before mcrt_source");
    if (!(L_erg_s > 0.0) || !isfinite(L_erg_s)) return fail(c, MCRT_EINVAL, "L_erg_s must be > 0");
    if (!pos_cm) return fail(c, MCRT_EINVAL, "pos_cm is NULL");
    const int n[3] = {c->nx, c->ny, c->nz};
    for (int a = 0; a < 3; ++a) {
        const double p = pos_cm[a] / c->h;
        if (!(p > 0.0) || !(p < (double)n[a])) return fail(c, MCRT_EINVAL, "source position must be strictly inside the grid");
        c->pos[a] = p;
    }
    std::vector<double> w(c->nf);
    if (T_star_K > 0.0) {
        for (int j = 0; j < c->nf; ++j) w[j] = planck_nu(c->nu[j], T_star_K) * c->dnu[j];
    } else {
        if (!L_nu_weights) return fail(c, MCRT_EINVAL, "T_star_K <= 0 needs L_nu_weights");
        double tot = 0.0;
        for (int j = 0; j < c->nf; ++j) {
            if (!(L_nu_weights[j] >= 0.0) || !isfinite(L_nu_weights[j])) return fail(c, MCRT_EINVAL, "L_nu_weights must be finite and >= 0");
            w[j] = L_nu_weights[j] * c->dnu[j];
            tot += w[j];
        }
        if (!(tot > 0.0)) return fail(c, MCRT_EINVAL, "L_nu_weights are all zero");
    }
    c->srccdf.resize(c->nf);
    make_cdf(w, c->srccdf.data());
    c->L = L_erg_s;
    CUDA_TRY(c, cudaMemcpyAsync(c->d_srccdf, c->srccdf.data(), (size_t)c->nf * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    {
        // Hot cells: the (at most hot_max) dusty cells whose centres lie nearest to the source, within 5.5 cells.
        int rc2;
        const size_t stage_words = 4 * (size_t)(kHot + 1) + 2 * 1400;
        if (!c->d_hot_idx && (rc2 = ws_alloc(c, (void **)&c->d_hot_idx, (kHot + 1 + stage_words + 2 * 1400) * sizeof(uint32_t)))) return rc2;
        uint32_t *d_stage = c->d_hot_idx + (kHot + 1);
        struct Cand { double d2; uint32_t idx; };
        std::vector<Cand> cand;
        const int sx = (int)floor(c->pos[0]), sy = (int)floor(c->pos[1]), sz = (int)floor(c->pos[2]);
        for (int iz = sz - 5; iz <= sz + 5; ++iz)
            for (int iy = sy - 5; iy <= sy + 5; ++iy)
                for (int ix = sx - 5; ix <= sx + 5; ++ix) {
                    if (ix < 0 || iy < 0 || iz < 0 || ix >= c->nx || iy >= c->ny || iz >= c->nz) continue;
                    const double dx = ix + 0.5 - c->pos[0], dy = iy + 0.5 - c->pos[1], dz = iz + 0.5 - c->pos[2];
                    const double d2 = dx * dx + dy * dy + dz * dz;
                    if (d2 <= 30.25) cand.push_back({d2, (uint32_t)((iz + kGuard) * c->pxy + (iy + kGuard) * c->px + (ix + kGuard))});
                }
        const int nc_ = (int)cand.size();      // <= 11^3 = 1331
        std::vector<unsigned long long> words(nc_);
        if (nc_) {
            std::vector<uint32_t> ci(nc_);
            for (int i = 0; i < nc_; ++i) ci[i] = cand[i].idx;
            unsigned long long *d_words = reinterpret_cast<unsigned long long *>(d_stage + 1400 + ((kHot + 1 + 1400) & 1));
            CUDA_TRY(c, cudaMemcpyAsync(d_stage, ci.data(), nc_ * 4, cudaMemcpyHostToDevice, c->stream));
            k_fetch_words<<<(nc_ + 127) / 128, 128, 0, c->stream>>>(c->cellw, d_stage, d_words, nc_);
            CUDA_TRY(c, cudaGetLastError());
            CUDA_TRY(c, cudaMemcpyAsync(words.data(), d_words, (size_t)nc_ * 8, cudaMemcpyDeviceToHost, c->stream));
            CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        }
        std::vector<Cand> dusty;
        for (int i = 0; i < nc_; ++i) {
            const uint32_t hi = (uint32_t)(words[i] >> 32);
            if (hi - 1u < 0x7FEFFFFFu) dusty.push_back(cand[i]);
        }
        std::stable_sort(dusty.begin(), dusty.end(), [](const Cand &a, const Cand &b) { return a.d2 < b.d2 || (a.d2 == b.d2 && a.idx < b.idx); });
        if ((int)dusty.size() > c->hot_max) dusty.resize(c->hot_max);
        // the previous source's numbering goes; the new one is written when a run knows how many cells it can hold
        if ((rc2 = apply_hot(c, 0))) return rc2;
        c->hot_cand.clear();
        for (const Cand &d : dusty) c->hot_cand.push_back(d.idx);
    }
    c->have_source = true;
    return MCRT_OK;
}

int mcrt_escape_bins(mcrt_ctx *c, int n_dir, const double *abs_mu_edges)
{
    if (!c) return MCRT_EINVAL;
    if (n_dir < 1 || n_dir > 4096 || !abs_mu_edges) return fail(c, MCRT_EINVAL, "n_dir must be in 1..4096");
    if (abs_mu_edges[0] != 0.0 || abs_mu_edges[n_dir] != 1.0) return fail(c, MCRT_EINVAL, "abs_mu_edges must run from 0 to 1");
    for (int b = 0; b < n_dir; ++b)
        if (!(abs_mu_edges[b + 1] > abs_mu_edges[b])) return fail(c, MCRT_EINVAL, "abs_mu_edges must be strictly ascending");
    c->ndir = n_dir;
    c->mu_edges.assign(abs_mu_edges, abs_mu_edges + n_dir + 1);
    c->mu_dirty = true;
    return MCRT_OK;
}

static int ensure_histograms(mcrt_ctx *c)
{
    if (c->mu_edges.empty()) { c->mu_edges = {0.0, 1.0}; c->ndir = 1; c->mu_dirty = true; }
    if (!c->mu_dirty) return MCRT_OK;
    int rc;
    if (c->ndir > c->ndir_alloc) {
        if ((rc = ws_alloc(c, (void **)&c->d_mu, (size_t)(c->ndir + 1) * 8))) return rc;
        if ((rc = ws_alloc(c, (void **)&c->sed, (size_t)c->ndir * c->nf * 8))) return rc;
        if ((rc = ws_alloc(c, (void **)&c->sed_direct, (size_t)c->ndir * c->nf * 8))) return rc;
        if ((rc = ws_alloc(c, (void **)&c->sed_stage, (size_t)c->ndir * c->nf * 8))) return rc;
        c->ndir_alloc = c->ndir;
    }
    CUDA_TRY(c, cudaMemcpyAsync(c->d_mu, c->mu_edges.data(), (size_t)(c->ndir + 1) * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->sed, 0, (size_t)c->ndir * c->nf * 8, c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->sed_direct, 0, (size_t)c->ndir * c->nf * 8, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));  // mu_edges.data() must outlive the copy
    c->mu_dirty = false;
    return MCRT_OK;
}

// the sixteen instantiations of the transport kernel
typedef void (*transport_fn)(const TransportParams);
// (digests recorded, hot cells tallied per CTA, level of the rarely used extras -- compiled out of the default kernels:
// the kernel's code has to fit the instruction cache, and every feature inlined into the event phase cost 1-4 % of the
// default path's throughput; the features that sit inside the walk loop halve it and have a level of their own)
static transport_fn transport_kernel(bool record, bool hot, int xtra)
{
#define MCRT_KT(x) k_transport<false, false, x>, k_transport<true, false, x>, k_transport<false, true, x>, k_transport<true, true, x>
    static const transport_fn tab[16] = {MCRT_KT(0), MCRT_KT(1), MCRT_KT(2), MCRT_KT(3)};
#undef MCRT_KT
    return tab[(record ? 1 : 0) | (hot ? 2 : 0) | (4 * xtra)];
}

static int transport_config(mcrt_ctx *c, const mcrt_run_opts *o, int *blocks, int *threads, size_t *smem, int *n_hot)
{
    const bool record = o && o->record_digests;
    *threads = (o && o->block_threads > 0) ? o->block_threads : MCRT_MAX_THREADS;
    if (*threads % 32 || *threads > MCRT_MAX_THREADS || *threads < 32)
        return fail(c, MCRT_EINVAL, "block_threads must be a multiple of 32 in 32.." + std::to_string(MCRT_MAX_THREADS));
    // as many warps (each with its packet pool) as fit beside the tables in the 196 KB carve-out
    while (*threads > 32 && transport_smem_bytes(c->ns, c->nf, c->ndir, c->mwords, *threads, record, 0) > kMaxTransportSmem) *threads -= 32;
    // up to two warps fewer if that gets from the 196 KB carve-out into the 164 KB one (torus512: 576 threads beside
    // 92 KB of L1 are 4.5 % faster than 640 beside 60 KB; within one carve-out a warp less costs 1-2.5 %)
    if (!(o && o->block_threads > 0) && smem_carveout(transport_smem_bytes(c->ns, c->nf, c->ndir, c->mwords, *threads, record, 0)) > 164 * 1024)
        for (int t = *threads - 32; t >= *threads - 64 && t >= 32; t -= 32)
            if (smem_carveout(transport_smem_bytes(c->ns, c->nf, c->ndir, c->mwords, t, record, 0)) <= 164 * 1024) { *threads = t; break; }
    const size_t base = transport_smem_bytes(c->ns, c->nf, c->ndir, c->mwords, *threads, record, 0);
    // ... and as many hot cells as the carve-out these need leaves room for (live B&W needs every count in global memory)
    int nh = (c->mix || c->subR || (o && (o->no_hot_cells || o->lucy_hybrid || o->mode == MCRT_MODE_LIVE_BW))) ? 0 : (int)c->hot_cand.size();
    const size_t cap = smem_carveout(base) - kSmemOverhead;
    while (nh > 0 && transport_smem_bytes(c->ns, c->nf, c->ndir, c->mwords, *threads, record, nh) > cap) --nh;
    if (nh < 8) nh = 0;
    *n_hot = nh;
    *smem = transport_smem_bytes(c->ns, c->nf, c->ndir, c->mwords, *threads, record, nh);
    if (*smem > 48 * 1024) {
        for (int v = 0; v < 16; ++v)
            CUDA_TRY(c, cudaFuncSetAttribute(transport_kernel(v & 1, v & 2, v >> 2), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem));
    }
    int nsm = 148, occ = 1;
    CUDA_TRY(c, cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->device));
    CUDA_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, transport_kernel(false, true, 3), *threads, *smem));
    if (occ < 1) return fail(c, MCRT_EINVAL, "transport kernel does not fit on an SM with these table sizes");
    c->occ_blocks = occ;
    *blocks = (o && o->grid_blocks > 0) ? o->grid_blocks : nsm * occ;  // persistent: every CTA resident
    return MCRT_OK;
}

int mcrt_launch_config(mcrt_ctx *c, int *grid_blocks, int *block_threads, size_t *smem_bytes)
{
    if (!c || !c->have_tables) return c ? fail(c, MCRT_ESTATE, "tables not set") : MCRT_EINVAL;
    int rc = ensure_histograms(c);
    if (rc) return rc;
    int b, t, nh; size_t s;
    if ((rc = transport_config(c, nullptr, &b, &t, &s, &nh))) return rc;
    if (grid_blocks) *grid_blocks = b;
    if (block_threads) *block_threads = t;
    if (smem_bytes) *smem_bytes = s;
    return MCRT_OK;
}

static int fill_stats(mcrt_ctx *c, mcrt_run_stats *st)
{
    unsigned long long h[CNT_N];
    CUDA_TRY(c, cudaMemcpyAsync(h, c->counters, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    fold_timing(c);
    memset(st, 0, sizeof(*st));
    st->transport_ms = c->transport_ms; st->update_ms = c->update_ms;
    st->packets = h[CNT_PACKETS]; st->crossings = h[CNT_CROSS]; st->dusty_crossings = h[CNT_DUSTY];
    st->scatterings = h[CNT_SCA]; st->absorptions = h[CNT_ABS]; st->direct_escapes = h[CNT_DIRECT];
    st->escapes = h[CNT_PACKETS];
    st->flights = h[CNT_PACKETS] + h[CNT_SCA] + h[CNT_ABS];
    st->lucy_adds = h[CNT_DUSTY] + h[CNT_SCA] + h[CNT_ABS];
    st->epochs = c->epochs; st->gpu_launches = c->launches;
    st->fx_bits = c->fx; st->overflow = h[CNT_OVERFLOW] ? 1 : 0;
    return MCRT_OK;
}

int mcrt_get_stats(mcrt_ctx *c, mcrt_run_stats *st)
{
    if (!c || !st) return MCRT_EINVAL;
    int rc = fill_stats(c, st);
    if (rc) return rc;
    return st->overflow ? fail(c, MCRT_EOVERFLOW, "a Lucy fixed-point tally exceeded 2^62") : MCRT_OK;
}

static void launch_transport(mcrt_ctx *c, const TransportParams &P)
{
    const mcrt_ctx::Run &R = c->run;
    transport_kernel(R.o.record_digests != 0, R.hot, R.xtra)<<<R.blocks, R.threads, R.smem, c->stream>>>(P);
}

static MixArrays mix_arrays(mcrt_ctx *c)
{
    MixArrays A;
    A.kcnt[0] = c->kabs_cnt; A.kcnt[1] = c->kcnt1; A.kprev[0] = c->kprev; A.kprev[1] = c->kprev1;
    A.lfx[0] = c->lfx; A.lfx[1] = c->lfx1; A.tidx1 = c->tidx1;
    A.ncomp = c->d_mx_ncomp; A.mat = c->d_mx_mat; A.frac = c->d_mx_frac;
    return A;
}

static void fill_params(mcrt_ctx *c, TransportParams &P)
{
    memset(&P, 0, sizeof(P));
    P.cellw = c->cellw; P.lfx = c->lfx; P.kcnt = c->kabs_cnt;
    P.kext_h = c->d_kext_h; P.kabs_fx = c->d_kabs_fx; P.albedo = c->d_albedo; P.g = c->d_g;
    P.srccdf = c->d_srccdf; P.mu_edges = c->d_mu;
    P.sed = c->sed; P.sed_direct = c->sed_direct; P.counters = c->counters;
    P.source_strata = c->run.o.source_strata; P.live_bw = c->run.o.mode == MCRT_MODE_LIVE_BW; P.J = c->d_J; P.cellfac = c->run.cellfac;
    P.sca_slot = c->sca_ev ? c->d_sca_slot : nullptr; P.sca_ev = c->sca_ev; P.sca_cap = c->sca_cap;
    P.hot_idx = c->d_hot_idx; P.hot_shift = c->hot_shift; P.hot_mask = c->hot_mask; P.tidx_mask = c->tidx_mask; P.n_hot = c->n_hot;
    if (c->mix) {
        P.lfx1 = c->lfx1; P.kcnt1 = c->kcnt1; P.tidx1 = c->tidx1; P.kabs1_fx = c->d_kabs1_fx;
        P.mx_thr = reinterpret_cast<const double2 *>(c->d_mx_thr); P.mx_mat = c->d_mx_mat;
    }
    P.redraw = c->run.o.tau_redraw_per_cell ? 1 : 0;
    P.subR = c->subR; P.sub_shift = c->sub_shift; P.sub_cellw = c->sub_cellw; P.sub_lfx = c->sub_lfx; P.sub_kcnt = c->sub_kcnt;
    P.sub_n = c->n_subcells; P.nc_grid = c->nc;
    if (c->run.o.lucy_hybrid) { P.kmax_diag = c->d_kmax_diag; P.two_fx = ldexp(1.0, c->fx); P.inv_two_fx = ldexp(1.0, -c->fx); }
    P.dig = c->run.o.record_digests ? c->dig : nullptr;
    P.dig_base = c->dig_base; P.dig_n = c->dig_n;
    P.nx = c->nx; P.ny = c->ny; P.nz = c->nz; P.ns = c->ns; P.nf = c->nf; P.nT = c->nT; P.ndir = c->ndir;
    P.nfs = c->nfs; P.perm = c->d_perm;
    P.nbx = c->nbx; P.nby = c->nby;
    P.vmask = c->vmask; P.vbox = c->vbox; P.bsh = c->msh; P.mwords = c->mwords; P.ncp = (uint32_t)c->ncp;
    P.lpx = c->px; P.lpxy = c->pxy; P.inv_lpx = 1.0 / (double)c->px; P.inv_lpxy = 1.0 / (double)c->pxy;
    P.px = c->pos[0]; P.py = c->pos[1]; P.pz = c->pos[2];
    P.seed_lo = (uint32_t)c->run.seed; P.seed_hi = (uint32_t)(c->run.seed >> 32);
}

// this part's slice [lo, hi) of an id range of `count` packets (every epoch is split the same way)
static void part_slice(const mcrt_run_opts &o, uint64_t count, uint64_t *lo, uint64_t *hi)
{
    const uint64_t R = o.part_count > 1 ? (uint64_t)o.part_count : 1u, r = o.part_count > 1 ? (uint64_t)o.part_index : 0u;
    *lo = (uint64_t)(((unsigned __int128)count * r) / R);
    *hi = (uint64_t)(((unsigned __int128)count * (r + 1)) / R);
}

// epoch schedule (reading Q19): B0 doubling (or growing by `growth`) up to Bmax
static void schedule_defaults(uint64_t n_packets, uint64_t *B0, uint64_t *Bmax, double *growth)
{
    if (*B0 == 0) { *B0 = 256; while (*B0 * 2 <= n_packets / 256) *B0 *= 2; }
    if (*Bmax == 0) *Bmax = (uint64_t)1 << 22;
    if (*Bmax < *B0) *Bmax = *B0;
    if (*growth == 0.0) *growth = 2.0;
}
static uint64_t next_epoch_size(uint64_t Bnom, uint64_t Bmax, double growth)
{
    // B_{e+1} = min(floor(B_e * growth), Bmax), never shrinking
    const double nb = floor((double)Bnom * growth);
    uint64_t nn = nb >= 1.8e19 ? Bmax : (uint64_t)nb;
    if (nn < Bnom) nn = Bnom;
    return nn > Bmax ? Bmax : nn;
}

int mcrt_epoch_schedule(uint64_t n_packets, uint64_t epoch_B0, uint64_t epoch_Bmax, double epoch_growth, uint64_t *sizes_out,
                        uint64_t max_epochs, uint64_t *n_epochs_out)
{
    if (n_packets < 1 || !n_epochs_out || (epoch_growth != 0.0 && !(epoch_growth >= 1.0))) return MCRT_EINVAL;
    schedule_defaults(n_packets, &epoch_B0, &epoch_Bmax, &epoch_growth);
    uint64_t done = 0, Bnom = epoch_B0, e = 0;
    while (done < n_packets) {
        const uint64_t Be = (n_packets - done < Bnom) ? n_packets - done : Bnom;
        if (sizes_out && e < max_epochs) sizes_out[e] = Be;
        done += Be; ++e;
        Bnom = next_epoch_size(Bnom, epoch_Bmax, epoch_growth);
    }
    *n_epochs_out = e;
    return MCRT_OK;
}

int mcrt_part_slice(uint64_t count, int part_index, int part_count, uint64_t *lo_out, uint64_t *hi_out)
{
    if (part_count < 1 || part_index < 0 || part_index >= part_count || !lo_out || !hi_out) return MCRT_EINVAL;
    *lo_out = (uint64_t)(((unsigned __int128)count * (uint64_t)part_index) / (uint64_t)part_count);
    *hi_out = (uint64_t)(((unsigned __int128)count * ((uint64_t)part_index + 1)) / (uint64_t)part_count);
    return MCRT_OK;
}

int mcrt_measure_read_bandwidth(size_t bytes, int repeats, double *gb_per_s_out)
{
    if (!gb_per_s_out || bytes < 4096 || repeats < 1) return MCRT_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return fail(nullptr, MCRT_ECUDA, "no CUDA device");
    void *buf = nullptr; unsigned long long *sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const size_t n16 = bytes / 16;
    cudaError_t err = cudaMalloc(&buf, n16 * 16);
    if (err == cudaSuccess) err = cudaMalloc((void **)&sink, 8);
    if (err == cudaSuccess) err = cudaMemset(buf, 1, n16 * 16);
    if (err == cudaSuccess) err = cudaEventCreate(&e0);
    if (err == cudaSuccess) err = cudaEventCreate(&e1);
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, 0);
    // a launch long enough (about a millisecond) that its start and end do not count, and few enough threads that
    // every one keeps eight loads in flight
    int blocks = nsm * 4;
    while (blocks > nsm && (size_t)blocks * 512 * 16 > n16) blocks -= nsm;
    const int passes = (int)std::min<size_t>(4096, std::max<size_t>(1, ((size_t)4 << 30) / (n16 * 16)));
    double best = 0.0;
    for (int r = 0; err == cudaSuccess && r < repeats + 2; ++r) {     // two warm-up launches
        cudaEventRecord(e0);
        k_read_probe<<<blocks, 512>>>((const uint4 *)buf, n16, passes, sink);
        cudaEventRecord(e1);
        err = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
        if (err == cudaSuccess && r >= 2 && ms > 0.f) { const double g = (double)passes * (double)(n16 * 16) / (ms * 1e-3) / 1e9; if (g > best) best = g; }
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf); cudaFree(sink);
    if (err != cudaSuccess) return fail(nullptr, MCRT_ECUDA, cudaGetErrorString(err));
    *gb_per_s_out = best;
    return MCRT_OK;
}

int mcrt_run_begin(mcrt_ctx *c, uint64_t n_packets, uint64_t seed, const mcrt_run_opts *opts)
{
    if (!c) return MCRT_EINVAL;
    if (c->run.active) return fail(c, MCRT_ESTATE, "a run is in progress: call mcrt_run_end first");
    if (!c->have_tables || !c->have_source) return fail(c, MCRT_ESTATE, "call mcrt_dust_tables and mcrt_source before mcrt_run");
    if (n_packets < 1) return fail(c, MCRT_EINVAL, "n_packets must be >= 1");
    mcrt_run_opts o;
    if (opts) o = *opts; else mcrt_default_opts(&o);
    if (o.mode != MCRT_MODE_BW_EPOCH && o.mode != MCRT_MODE_FROZEN_T_SWEEP && o.mode != MCRT_MODE_LIVE_BW) return fail(c, MCRT_EINVAL, "unknown mode");
    if (o.mode == MCRT_MODE_LIVE_BW && o.part_count > 1) return fail(c, MCRT_EINVAL, "MCRT_MODE_LIVE_BW is not available in a partitioned run");
    if (o.mode == MCRT_MODE_FROZEN_T_SWEEP && o.n_sweeps < 1) return fail(c, MCRT_EINVAL, "n_sweeps must be >= 1");
    if (o.part_count < 0 || o.part_count > 65536 || (o.part_count > 1 && (o.part_index < 0 || o.part_index >= o.part_count)))
        return fail(c, MCRT_EINVAL, "part_index must be in 0..part_count-1");
    if (o.part_count <= 1) { o.part_count = 1; o.part_index = 0; }
    if (o.epoch_growth == 0.0) o.epoch_growth = 2.0;
    if (o.carry_interactions > 65535u) return fail(c, MCRT_EINVAL, "carry_interactions must be <= 65535");
    if (o.carry_interactions && o.part_count > 1) return fail(c, MCRT_EINVAL, "carry_interactions is not available in a partitioned run");
    if (!(o.epoch_growth >= 1.0) || !isfinite(o.epoch_growth)) return fail(c, MCRT_EINVAL, "epoch_growth must be >= 1");
    if (o.n_total && o.n_total < n_packets) return fail(c, MCRT_EINVAL, "n_total must be >= n_packets");
    if (o.first_packet_id + n_packets < o.first_packet_id) return fail(c, MCRT_EINVAL, "packet ids overflow 64 bits");
    if (c->mix && (o.mode == MCRT_MODE_LIVE_BW || o.part_count > 1))
        return fail(c, MCRT_EINVAL, "dust mixtures are not available in live B&W or partitioned runs");
    if (c->subR && (o.carry_interactions || o.lucy_hybrid || o.mode == MCRT_MODE_LIVE_BW || o.part_count > 1))
        return fail(c, MCRT_EINVAL, "grids with sub-cubes: no carry-over, thresholded estimator, live B&W or partitioned runs");
    if (o.tau_redraw_per_cell && (o.carry_interactions || o.mode == MCRT_MODE_LIVE_BW))
        return fail(c, MCRT_EINVAL, "tau_redraw_per_cell is not available with carry-over or in live B&W");
    if (o.lucy_hybrid && (c->mix || o.mode == MCRT_MODE_LIVE_BW || o.part_count > 1))
        return fail(c, MCRT_EINVAL, "lucy_hybrid is not available with mixtures, in live B&W or partitioned runs");
    if ((o.mode == MCRT_MODE_FROZEN_T_SWEEP || !o.reset_tallies) && c->last_n != 0 && c->hybrid != (o.lucy_hybrid != 0))
        return fail(c, MCRT_ESTATE, "the stored tallies were made with the other Lucy estimator (lucy_hybrid)");
    int rc = ensure_histograms(c);
    if (rc) return rc;
    if (o.lucy_hybrid && !c->d_kmax_diag) {
        std::vector<double> km(c->ns, 0.0);     // reading Q37: the diagonal at the frequency of the largest extinction
        for (int s_ = 0; s_ < c->ns; ++s_) {
            for (int j = 0; j < c->nf; ++j) km[s_] = fmax(km[s_], c->kabs[(size_t)s_ * c->nf + j] + c->ksca[(size_t)s_ * c->nf + j]);
            km[s_] = sqrt(3.0) * c->h * km[s_];
        }
        if (cudaMalloc((void **)&c->d_kmax_diag, c->ns * 8) != cudaSuccess) return fail(c, MCRT_ENOMEM, "cudaMalloc failed");
        CUDA_TRY(c, cudaMemcpy(c->d_kmax_diag, km.data(), c->ns * 8, cudaMemcpyHostToDevice));
    }
    mcrt_ctx::Run &R = c->run;
    int n_hot = 0;
    if ((rc = transport_config(c, &o, &R.blocks, &R.threads, &R.smem, &n_hot))) return rc;
    if ((rc = apply_hot(c, n_hot))) return rc;
    R.xtra = o.tau_redraw_per_cell ? 3 : (c->mix || o.lucy_hybrid) ? 2
             : ((o.carry_interactions || c->sca_ev || o.source_strata || o.mode == MCRT_MODE_LIVE_BW || c->subR) ? 1 : 0);
    R.hot = c->n_hot > 0;
    const size_t hist_bytes = (size_t)c->ndir * c->nf * 8;

    const uint64_t n_xi = o.n_total ? o.n_total : n_packets;
    const int fx = fx_bits_for(n_xi);
    const double xi = c->L / (double)n_xi;                          // xi = L/N
    const bool continuing = o.mode != MCRT_MODE_FROZEN_T_SWEEP && !o.reset_tallies && c->last_n != 0;
    if (continuing && (xi != c->xi || fx != c->fx))
        return fail(c, MCRT_ESTATE, "reset_tallies = 0: the stored tallies have another packet energy / fixed-point scale (set n_total)");
    if (continuing && c->globalised)
        return fail(c, MCRT_ESTATE, "reset_tallies = 0 after a partitioned run: the stored tallies are sums over the parts");

    if (o.record_digests) {
        if (c->dig_cap < n_packets) {
            if ((rc = ws_alloc(c, (void **)&c->dig, n_packets * sizeof(mcrt_digest)))) return rc;
            c->dig_cap = n_packets;
        }
        c->dig_n = n_packets;
        if (o.part_count > 1) CUDA_TRY(c, cudaMemsetAsync(c->dig, 0, n_packets * sizeof(mcrt_digest), c->stream));
    } else c->dig_n = 0;
    c->dig_base = o.first_packet_id;

    if (o.reset_tallies && o.mode != MCRT_MODE_FROZEN_T_SWEEP) {
        CUDA_TRY(c, cudaMemset2DAsync(c->lfx, 8 * kCS, 0, 8, c->ncp, c->stream));
        CUDA_TRY(c, cudaMemsetAsync(c->kabs_cnt, 0, c->ncp * 8, c->stream));
        CUDA_TRY(c, cudaMemsetAsync(c->kprev, 0, c->ncp * 8, c->stream));
        if (c->subR) {
            CUDA_TRY(c, cudaMemsetAsync(c->sub_lfx, 0, c->n_subcells * (size_t)kCS * 8, c->stream));
            CUDA_TRY(c, cudaMemsetAsync(c->sub_kcnt, 0, c->n_subcells * 8, c->stream));
            CUDA_TRY(c, cudaMemsetAsync(c->sub_kprev, 0, c->n_subcells * 8, c->stream));
        }
        if (c->mix) {
            CUDA_TRY(c, cudaMemsetAsync(c->lfx1, 0, c->ncp * (size_t)kCS * 8, c->stream));
            CUDA_TRY(c, cudaMemsetAsync(c->kcnt1, 0, c->ncp * 8, c->stream));
            CUDA_TRY(c, cudaMemsetAsync(c->kprev1, 0, c->ncp * 8, c->stream));
        }
        CUDA_TRY(c, cudaMemsetAsync(c->sed, 0, hist_bytes, c->stream));
        CUDA_TRY(c, cudaMemsetAsync(c->sed_direct, 0, hist_bytes, c->stream));
        CUDA_TRY(c, cudaMemsetAsync(c->counters, 0, CNT_N * 8, c->stream));
        c->epochs = 0; c->launches = 0;
        if (c->ev_used) { cudaStreamSynchronize(c->stream); fold_timing(c); }
        c->transport_ms = 0.0; c->update_ms = 0.0;
        c->globalised = false;
    }
    // Eq. 4 for the first sweep: the stored k and L are in packets of the run that made them
    R.prev_fx = c->fx;
    R.prev_cellfac = c->xi / (kFourPi * c->h * c->h * c->h);
    c->fx = fx; c->xi = xi;
    c->hybrid = o.lucy_hybrid != 0;
    R.cellfac = xi / (kFourPi * c->h * c->h * c->h);             // xi / (4 pi V) of Eq. 4
    c->last_n = n_packets;
    {
        const size_t nsf = (size_t)c->ns * c->nf;
        std::vector<double> kfx(nsf);
        for (size_t i = 0; i < nsf; ++i) kfx[i] = ldexp(c->kabs_h[i], c->fx);
        CUDA_TRY(c, cudaMemcpyAsync(c->d_kabs_fx, kfx.data(), nsf * 8, cudaMemcpyHostToDevice, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        if (c->mix) {
            for (size_t i = 0; i < nsf; ++i) kfx[i] = ldexp(c->kabs1_h[i], c->fx);
            CUDA_TRY(c, cudaMemcpyAsync(c->d_kabs1_fx, kfx.data(), nsf * 8, cudaMemcpyHostToDevice, c->stream));
            CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        }
    }
    const size_t j_smem = (size_t)c->ns * c->nT * 8;
    if (j_smem > 48 * 1024) {
        CUDA_TRY(c, cudaFuncSetAttribute(k_epoch_update, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)j_smem));
        CUDA_TRY(c, cudaFuncSetAttribute(k_sweep_update, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)j_smem));
        CUDA_TRY(c, cudaFuncSetAttribute(k_mix_update, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)j_smem));
        CUDA_TRY(c, cudaFuncSetAttribute(k_hybrid_update, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)j_smem));
    }
    R.o = o; R.n = n_packets; R.seed = seed; R.done = 0; R.Bprev = 0; R.e = 0; R.sweep = 0; R.finished = false;
    R.carry_K = (o.mode == MCRT_MODE_BW_EPOCH) ? o.carry_interactions : 0u; R.n_carry = 0;
    R.growth = o.epoch_growth;
    uint64_t B0 = o.epoch_B0, Bmax = o.epoch_Bmax;
    if (o.mode == MCRT_MODE_LIVE_BW) B0 = Bmax = n_packets;      // one launch: nothing is frozen per epoch
    schedule_defaults(n_packets, &B0, &Bmax, &R.growth);
    R.Bnom = B0; R.Bmax = Bmax;
    c->need_exchange = false; c->exchange_open = false;
    R.active = true;
    return MCRT_OK;
}

int mcrt_run_step(mcrt_ctx *c, int *done_out)
{
    if (!c) return MCRT_EINVAL;
    mcrt_ctx::Run &R = c->run;
    if (!R.active) return fail(c, MCRT_ESTATE, "mcrt_run_step without mcrt_run_begin");
    if (c->need_exchange) return fail(c, MCRT_ESTATE, "partitioned run: the parts' tallies must be exchanged after every step");
    if (R.finished) { if (done_out) *done_out = 1; return MCRT_OK; }
    const mcrt_run_opts &o = R.o;
    const bool timing = o.time_kernels != 0;
    const size_t j_smem = (size_t)c->ns * c->nT * 8;
    const int ugrid = stream_grid(c->ncp);
    const size_t hist_bytes = (size_t)c->ndir * c->nf * 8;
    TransportParams P;
    fill_params(c, P);
    uint64_t lo, hi;
    if (o.mode != MCRT_MODE_FROZEN_T_SWEEP) {
        // an epoch of new packets, or -- all new packets done, some still carried -- an epoch of carried packets only,
        // with the budget doubled (see CarryRec)
        const bool drain = R.done >= R.n;
        const uint64_t Be = drain ? 0 : ((R.n - R.done < R.Bnom) ? R.n - R.done : R.Bnom);
        if (drain) R.carry_K = R.carry_K > 0x40000000u ? 0x80000000u : 2u * R.carry_K;
        P.cdf = c->d_cdfdB;
        P.pass = o.rng_pass;
        if (R.carry_K) {
            // room for every packet of this epoch in the list it may leave behind
            const int out = c->carry_cur ^ 1;
            const size_t need = (size_t)(R.n_carry + Be);
            if (c->carry_cap[out] < need) {
                if (c->carry_buf[out]) { CUDA_TRY(c, cudaStreamSynchronize(c->stream)); cudaFree(c->carry_buf[out]); c->carry_buf[out] = nullptr; c->carry_cap[out] = 0; }
                const size_t cap = need + need / 4 + 1024;
                if (cudaMalloc((void **)&c->carry_buf[out], cap * sizeof(CarryRec)) != cudaSuccess)
                    return fail(c, MCRT_ENOMEM, "cudaMalloc of the carry-over list failed");
                c->carry_cap[out] = cap;
            }
            P.carry_in = c->carry_buf[c->carry_cur]; P.carry_out = c->carry_buf[out];
            P.n_carry_in = (uint32_t)R.n_carry; P.carry_K = R.carry_K;
        }
        mark(c, timing);
        if (o.lucy_hybrid)
            k_hybrid_update<<<ugrid, 256, j_smem, c->stream>>>(c->cellw, c->kabs_cnt, c->kprev, c->lfx, c->d_J, c->d_kmax_diag, c->nT,
                                                              c->ns, c->ncp, 0, R.e == 0,
                                                              (R.e == 0 || drain) ? 1.0 : (double)Be / (double)R.Bprev,
                                                              ldexp(1.0, -c->fx), R.cellfac, c->counters, c->tidx_mask);
        else if (c->mix)
            k_mix_update<<<ugrid, 256, j_smem, c->stream>>>(c->cellw, mix_arrays(c), c->d_J, c->nT, c->ns, c->ncp, 0, R.e == 0,
                                                           (R.e == 0 || drain) ? 1.0 : (double)Be / (double)R.Bprev, 0, 0.0,
                                                           R.cellfac, c->counters, c->tidx_mask);
        else
        k_epoch_update<<<ugrid, 256, j_smem, c->stream>>>(c->cellw, c->kabs_cnt, c->kprev, c->lfx, c->d_J, c->nT, c->ns, c->ncp,
                                                         R.e == 0, (R.e == 0 || drain) ? 1.0 : (double)Be / (double)R.Bprev,
                                                         R.cellfac, c->counters, c->tidx_mask);
        if (c->subR)    // the sub-cubes: the same rule, Eq. 4 with V = (h/R)^3
            k_epoch_update<<<stream_grid(c->n_subcells), 256, j_smem, c->stream>>>(c->sub_cellw, c->sub_kcnt, c->sub_kprev, c->sub_lfx, c->d_J,
                                                                                  c->nT, c->ns, c->n_subcells, R.e == 0,
                                                                                  (R.e == 0 || drain) ? 1.0 : (double)Be / (double)R.Bprev,
                                                                                  R.cellfac * (double)(c->subR * c->subR * c->subR), c->counters,
                                                                                  c->tidx_mask);
        part_slice(o, Be, &lo, &hi);
        P.pid0 = o.first_packet_id + R.done + lo; P.count = hi - lo;
        mark(c, timing);
        if (P.count + P.n_carry_in) {
            launch_transport(c, P);
        }
        mark(c, timing);
        c->launches += (P.count + P.n_carry_in) ? 2 : 1;
        c->epochs++;
        if (!drain) {
            R.done += Be; R.Bprev = Be;
            R.Bnom = next_epoch_size(R.Bnom, R.Bmax, R.growth);
        }
        ++R.e;
        if (R.carry_K) {
            // how many packets were carried over: needed to size the next launch (8-byte read, synchronises)
            unsigned long long nc_ = 0ull;
            CUDA_TRY(c, cudaMemcpyAsync(&nc_, c->counters + CNT_CARRY, 8, cudaMemcpyDeviceToHost, c->stream));
            CUDA_TRY(c, cudaStreamSynchronize(c->stream));
            R.n_carry = nc_;
            c->carry_cur ^= 1;
        }
        R.finished = R.done >= R.n && R.n_carry == 0;
    } else {
        const int sw = ++R.sweep;
        P.cdf = c->d_cdfB;
        // temperatures of the previous pass (its own packet energy and fixed-point scale), then zero and re-run all N packets
        mark(c, timing);
        if (o.lucy_hybrid)
            k_hybrid_update<<<ugrid, 256, j_smem, c->stream>>>(c->cellw, c->kabs_cnt, c->kprev, c->lfx, c->d_J, c->d_kmax_diag, c->nT,
                                                              c->ns, c->ncp, 1, 0, 1.0, ldexp(1.0, -(sw == 1 ? R.prev_fx : c->fx)),
                                                              sw == 1 ? R.prev_cellfac : R.cellfac, c->counters, c->tidx_mask);
        else if (c->mix)
            k_mix_update<<<ugrid, 256, j_smem, c->stream>>>(c->cellw, mix_arrays(c), c->d_J, c->nT, c->ns, c->ncp, 1, 0, 1.0,
                                                           o.sweep_T_from_lucy, ldexp(1.0, -(sw == 1 ? R.prev_fx : c->fx)),
                                                           sw == 1 ? R.prev_cellfac : R.cellfac, c->counters, c->tidx_mask);
        else
        k_sweep_update<<<ugrid, 256, j_smem, c->stream>>>(c->cellw, c->kabs_cnt, c->kprev, c->lfx, c->d_J, c->nT, c->ns, c->ncp,
                                                         o.sweep_T_from_lucy, ldexp(1.0, -(sw == 1 ? R.prev_fx : c->fx)),
                                                         sw == 1 ? R.prev_cellfac : R.cellfac, c->counters, c->tidx_mask);
        if (c->subR)
            k_sweep_update<<<stream_grid(c->n_subcells), 256, j_smem, c->stream>>>(c->sub_cellw, c->sub_kcnt, c->sub_kprev, c->sub_lfx, c->d_J,
                                                                                  c->nT, c->ns, c->n_subcells, o.sweep_T_from_lucy,
                                                                                  ldexp(1.0, -(sw == 1 ? R.prev_fx : c->fx)),
                                                                                  (sw == 1 ? R.prev_cellfac : R.cellfac) * (double)(c->subR * c->subR * c->subR),
                                                                                  c->counters, c->tidx_mask);
        CUDA_TRY(c, cudaMemsetAsync(c->sed, 0, hist_bytes, c->stream));
        CUDA_TRY(c, cudaMemsetAsync(c->sed_direct, 0, hist_bytes, c->stream));
        CUDA_TRY(c, cudaMemsetAsync(c->counters, 0, CNT_NEXT * 8, c->stream));
        CUDA_TRY(c, cudaMemsetAsync(c->counters + CNT_SCAEV, 0, 8, c->stream));   // every sweep starts an empty event list
        c->globalised = false;
        if (o.part_count > 1 && o.record_digests) CUDA_TRY(c, cudaMemsetAsync(c->dig, 0, c->dig_n * sizeof(mcrt_digest), c->stream));
        P.pass = o.rng_pass + (uint32_t)sw;
        part_slice(o, R.n, &lo, &hi);
        P.pid0 = o.first_packet_id + lo; P.count = hi - lo;
        mark(c, timing);
        if (P.count) {
            launch_transport(c, P);
        }
        mark(c, timing);
        c->launches += P.count ? 2 : 1;
        c->epochs++;
        R.finished = sw >= o.n_sweeps;
    }
    CUDA_TRY(c, cudaGetLastError());
    if (o.part_count > 1) {
        c->need_exchange = true;
        c->exchange_full = R.finished || o.mode == MCRT_MODE_FROZEN_T_SWEEP;
    }
    if (done_out) *done_out = R.finished ? 1 : 0;
    return MCRT_OK;
}

int mcrt_run_end(mcrt_ctx *c, mcrt_run_stats *stats_out)
{
    if (!c) return MCRT_EINVAL;
    mcrt_ctx::Run &R = c->run;
    if (!R.active) return fail(c, MCRT_ESTATE, "mcrt_run_end without mcrt_run_begin");
    if (!R.finished) return fail(c, MCRT_ESTATE, "mcrt_run_end before the last mcrt_run_step");
    if (c->need_exchange) return fail(c, MCRT_ESTATE, "partitioned run: exchange the last step's tallies before mcrt_run_end");
    k_range_check<<<stream_grid(c->ncp), 256, 0, c->stream>>>(c->lfx, c->ncp, c->counters);
    if (c->mix) k_range_check<<<stream_grid(c->ncp), 256, 0, c->stream>>>(c->lfx1, c->ncp, c->counters);
    if (c->subR) k_range_check<<<stream_grid(c->n_subcells), 256, 0, c->stream>>>(c->sub_lfx, c->n_subcells, c->counters);
    c->launches += c->mix ? 2 : 1;
    R.active = false;
    CUDA_TRY(c, cudaGetLastError());
    if (stats_out) {
        int rc;
        if ((rc = fill_stats(c, stats_out))) return rc;
        if (stats_out->overflow) return fail(c, MCRT_EOVERFLOW, "a Lucy fixed-point tally exceeded 2^62");
    }
    return MCRT_OK;
}

int mcrt_run(mcrt_ctx *c, uint64_t n_packets, uint64_t seed, const mcrt_run_opts *opts, mcrt_run_stats *stats_out)
{
    if (!c) return MCRT_EINVAL;
    if (opts && opts->part_count > 1)
        return fail(c, MCRT_EINVAL, "a partitioned run needs an exchange after every step: use mcrt_run_begin / _step / _end");
    int rc = mcrt_run_begin(c, n_packets, seed, opts);
    if (rc) return rc;
    int done = 0;
    while (!done)
        if ((rc = mcrt_run_step(c, &done))) { c->run.active = false; return rc; }
    return mcrt_run_end(c, stats_out);
}

int mcrt_exchange_begin(mcrt_ctx *c, mcrt_exchange *out)
{
    if (!c || !out) return MCRT_EINVAL;
    if (!c->need_exchange || c->exchange_open) return fail(c, MCRT_ESTATE, "mcrt_exchange_begin: no step of a partitioned run is waiting for its exchange");
    memset(out, 0, sizeof(*out));
    // this epoch's own increments k - k_prev (k_prev = the global counts the epoch started from)
    k_count_delta<<<stream_grid(c->ncp), 256, 0, c->stream>>>(c->kabs_cnt, c->kprev, c->ncp, 0);
    c->launches += 1;
    CUDA_TRY(c, cudaGetLastError());
    int n = 0;
    out->ptr[n] = c->kabs_cnt; out->words[n++] = c->ncp;
    if (c->exchange_full) {
        if (kCS == 1) out->ptr[n] = c->lfx;
        else {   // the tallies sit in the cell records: exchanged through a contiguous staging copy
            k_lucy_stage<<<stream_grid(c->ncp), 256, 0, c->stream>>>(c->lfx, (long long *)c->scratch, c->ncp, 0);
            c->launches += 1;
            out->ptr[n] = c->scratch;
        }
        out->words[n++] = c->ncp;
        out->ptr[n] = c->sed; out->words[n++] = (uint64_t)c->ndir * c->nf;
        out->ptr[n] = c->sed_direct; out->words[n++] = (uint64_t)c->ndir * c->nf;
        out->ptr[n] = c->counters; out->words[n++] = CNT_NEXT;
        if (c->dig_n) { out->ptr[n] = c->dig; out->words[n++] = c->dig_n * (sizeof(mcrt_digest) / 8); }  // zero except own packets
    }
    out->n = n;
    c->exchange_open = true;
    return MCRT_OK;
}

int mcrt_exchange_end(mcrt_ctx *c)
{
    if (!c) return MCRT_EINVAL;
    if (!c->exchange_open) return fail(c, MCRT_ESTATE, "mcrt_exchange_end without mcrt_exchange_begin");
    k_count_delta<<<stream_grid(c->ncp), 256, 0, c->stream>>>(c->kabs_cnt, c->kprev, c->ncp, 1);
    c->launches += 1;
    if (c->exchange_full && kCS != 1) {
        k_lucy_stage<<<stream_grid(c->ncp), 256, 0, c->stream>>>(c->lfx, (long long *)c->scratch, c->ncp, 1);
        c->launches += 1;
    }
    CUDA_TRY(c, cudaGetLastError());
    if (c->exchange_full) c->globalised = true;
    c->exchange_open = false;
    c->need_exchange = false;
    return MCRT_OK;
}

int mcrt_exchange_peer_sum(mcrt_ctx *c, int part_index, int n_parts, const mcrt_exchange *views, int phase)
{
    if (!c || !views) return MCRT_EINVAL;
    if (n_parts < 1 || n_parts > kMaxParts || part_index < 0 || part_index >= n_parts || (phase != 0 && phase != 1))
        return fail(c, MCRT_EINVAL, "mcrt_exchange_peer_sum: 1 <= n_parts <= 16, 0 <= part_index < n_parts, phase 0 or 1");
    for (int q = 1; q < n_parts; ++q) {
        if (views[q].n != views[0].n) return fail(c, MCRT_EINVAL, "mcrt_exchange_peer_sum: the parts list different arrays");
        for (int a = 0; a < views[0].n; ++a)
            if (views[q].words[a] != views[0].words[a]) return fail(c, MCRT_EINVAL, "mcrt_exchange_peer_sum: array lengths differ between parts");
    }
    for (int a = 0; a < views[0].n; ++a) {
        PeerPtrs pp;
        for (int q = 0; q < kMaxParts; ++q) pp.p[q] = (unsigned long long *)views[q < n_parts ? q : 0].ptr[a];
        const size_t words = views[0].words[a];
        k_peer_sum<<<stream_grid(phase == 0 ? (words + n_parts - 1) / n_parts : words), 256, 0, c->stream>>>(pp, part_index, n_parts, words, phase);
        c->launches += 1;
    }
    CUDA_TRY(c, cudaGetLastError());
    return MCRT_OK;
}

int mcrt_exchange_local(mcrt_ctx *const *parts, int n_parts)
{
    if (!parts || n_parts < 1 || n_parts > kMaxParts) return MCRT_EINVAL;
    std::vector<mcrt_exchange> v(n_parts);
    int rc;
    for (int q = 0; q < n_parts; ++q) {
        if (!parts[q]) return MCRT_EINVAL;
        if ((rc = mcrt_exchange_begin(parts[q], &v[q]))) return rc;
    }
    // one device, possibly several streams: every part's step must have finished before anyone reads its tallies
    for (int phase = 0; phase < 2; ++phase) {
        for (int q = 0; q < n_parts; ++q) CUDA_TRY(parts[q], cudaStreamSynchronize(parts[q]->stream));
        for (int q = 0; q < n_parts; ++q)
            if ((rc = mcrt_exchange_peer_sum(parts[q], q, n_parts, v.data(), phase))) return rc;
    }
    for (int q = 0; q < n_parts; ++q) CUDA_TRY(parts[q], cudaStreamSynchronize(parts[q]->stream));
    for (int q = 0; q < n_parts; ++q)
        if ((rc = mcrt_exchange_end(parts[q]))) return rc;
    return MCRT_OK;
}

static int gather_out(mcrt_ctx *c, int what, void *dst, size_t elem, mcrt_mem where, int comp = 0)
{
    if (!dst) return MCRT_OK;
    void *dev = (where == MCRT_DEVICE) ? dst : c->scratch;
    const double cellfac = c->xi / (kFourPi * c->h * c->h * c->h);
    k_gather<<<stream_grid(c->nc), 256, 0, c->stream>>>(what, dev, c->cellw, comp ? c->kcnt1 : c->kabs_cnt, comp ? c->lfx1 : c->lfx,
                                                       c->d_J, c->d_Tg, c->nT, c->nx, c->ny, c->nz, c->px, c->pxy, c->xi,
                                                       ldexp(1.0, -c->fx), cellfac, c->tidx_mask, c->mix ? c->d_mx_mat : nullptr,
                                                       c->d_mx_frac, comp, c->tidx1, c->d_kmax_diag);
    CUDA_TRY(c, cudaGetLastError());
    if (where == MCRT_HOST) {
        CUDA_TRY(c, cudaMemcpyAsync(dst, dev, c->nc * elem, cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    }
    return MCRT_OK;
}

// the read calls refuse to hand back wrapped tallies (the flag is set by the per-epoch update and the final range check)
static int check_overflow(mcrt_ctx *c)
{
    unsigned long long flag = 0ull;
    CUDA_TRY(c, cudaMemcpyAsync(&flag, c->counters + CNT_OVERFLOW, 8, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return flag ? fail(c, MCRT_EOVERFLOW, "a Lucy fixed-point tally exceeded 2^62") : MCRT_OK;
}

int mcrt_read(mcrt_ctx *c, double *E_abs_count, double *E_abs_lucy, float *T_count, float *T_lucy, double *SED, mcrt_mem where)
{
    if (!c) return MCRT_EINVAL;
    if (!c->last_n) return fail(c, MCRT_ESTATE, "mcrt_read before mcrt_run");
    if (c->run.active) return fail(c, MCRT_ESTATE, "mcrt_read inside mcrt_run_begin .. mcrt_run_end");
    int rc;
    if ((rc = check_overflow(c))) return rc;
    if ((rc = gather_out(c, G_ECOUNT, E_abs_count, 8, where))) return rc;
    if ((rc = gather_out(c, G_ELUCY, E_abs_lucy, 8, where))) return rc;
    if ((rc = gather_out(c, G_TCOUNT, T_count, 4, where))) return rc;
    if ((rc = gather_out(c, c->hybrid ? G_THYBRID : G_TLUCY, T_lucy, 4, where))) return rc;
    if (SED) {
        const int n = c->ndir * c->nf;
        double *dev = (where == MCRT_DEVICE) ? SED : c->sed_stage;
        k_sed<<<(n + 255) / 256, 256, 0, c->stream>>>(dev, c->sed, c->d_dnu, c->d_mu, c->ndir, c->nf, c->xi);
        CUDA_TRY(c, cudaGetLastError());
        if (where == MCRT_HOST) {
            CUDA_TRY(c, cudaMemcpyAsync(SED, dev, (size_t)n * 8, cudaMemcpyDeviceToHost, c->stream));
        }
    }
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MCRT_OK;
}

int mcrt_read_component(mcrt_ctx *c, int component, double *E_abs_count, double *E_abs_lucy, float *T_count, float *T_lucy,
                        uint64_t *k_abs, int64_t *lucy_fx, uint16_t *tidx, mcrt_mem where)
{
    if (!c) return MCRT_EINVAL;
    if (!c->mix) return fail(c, MCRT_ESTATE, "mcrt_read_component without mcrt_dust_mixtures");
    if (component < 0 || component > 1) return fail(c, MCRT_EINVAL, "component must be 0 or 1");
    if (!c->last_n) return fail(c, MCRT_ESTATE, "mcrt_read_component before mcrt_run");
    if (c->run.active) return fail(c, MCRT_ESTATE, "mcrt_read_component inside mcrt_run_begin .. mcrt_run_end");
    int rc;
    if ((rc = check_overflow(c))) return rc;
    if ((rc = gather_out(c, G_ECOUNT, E_abs_count, 8, where, component))) return rc;
    if ((rc = gather_out(c, G_ELUCY, E_abs_lucy, 8, where, component))) return rc;
    if ((rc = gather_out(c, G_TCOUNT, T_count, 4, where, component))) return rc;
    if ((rc = gather_out(c, G_TLUCY, T_lucy, 4, where, component))) return rc;
    if ((rc = gather_out(c, G_K, k_abs, 8, where, component))) return rc;
    if ((rc = gather_out(c, G_LFX, lucy_fx, 8, where, component))) return rc;
    if ((rc = gather_out(c, G_TIDX, tidx, 2, where, component))) return rc;
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MCRT_OK;
}

int mcrt_read_raw(mcrt_ctx *c, uint64_t *k_abs, int64_t *lucy_fx, uint64_t *sed_counts, uint64_t *sed_direct, uint16_t *tidx,
                  mcrt_digest *digests, mcrt_mem where)
{
    if (!c) return MCRT_EINVAL;
    if (!c->last_n) return fail(c, MCRT_ESTATE, "mcrt_read_raw before mcrt_run");
    int rc;
    if ((rc = check_overflow(c))) return rc;
    if ((rc = gather_out(c, G_K, k_abs, 8, where))) return rc;
    if ((rc = gather_out(c, G_LFX, lucy_fx, 8, where))) return rc;
    if ((rc = gather_out(c, G_TIDX, tidx, 2, where))) return rc;
    const cudaMemcpyKind kind = (where == MCRT_HOST) ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
    const size_t hb = (size_t)c->ndir * c->nf * 8;
    if (sed_counts) CUDA_TRY(c, cudaMemcpyAsync(sed_counts, c->sed, hb, kind, c->stream));
    if (sed_direct) CUDA_TRY(c, cudaMemcpyAsync(sed_direct, c->sed_direct, hb, kind, c->stream));
    if (digests) {
        if (!c->dig_n) return fail(c, MCRT_ESTATE, "digests were not recorded by the last run");
        CUDA_TRY(c, cudaMemcpyAsync(digests, c->dig, c->dig_n * sizeof(mcrt_digest), kind, c->stream));
    }
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MCRT_OK;
}

int mcrt_scatter_store(mcrt_ctx *c, int n_bins, const int32_t *nu_bins, uint64_t capacity)
{
    if (!c) return MCRT_EINVAL;
    if (!c->have_tables) return fail(c, MCRT_ESTATE, "call mcrt_dust_tables before mcrt_scatter_store");
    if (c->run.active) return fail(c, MCRT_ESTATE, "mcrt_scatter_store inside a run");
    if (n_bins < 1 || n_bins > 16 || !nu_bins || capacity < 1) return fail(c, MCRT_EINVAL, "1 <= n_bins <= 16, capacity >= 1");
    std::vector<int8_t> slot(c->nf, (int8_t)-1);
    for (int b = 0; b < n_bins; ++b) {
        if (nu_bins[b] < 0 || nu_bins[b] >= c->nf) return fail(c, MCRT_EINVAL, "nu_bins out of range");
        slot[nu_bins[b]] = (int8_t)b;
    }
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    if (c->sca_ev) { cudaFree(c->sca_ev); c->sca_ev = nullptr; c->sca_cap = 0; }
    if (!c->d_sca_slot && cudaMalloc((void **)&c->d_sca_slot, c->nf) != cudaSuccess) return fail(c, MCRT_ENOMEM, "cudaMalloc failed");
    if (cudaMalloc((void **)&c->sca_ev, capacity * sizeof(mcrt_scatter_event)) != cudaSuccess)
        return fail(c, MCRT_ENOMEM, "cudaMalloc of the scattering-event list failed");
    c->sca_cap = capacity;
    c->sca_bins.assign(nu_bins, nu_bins + n_bins);
    CUDA_TRY(c, cudaMemcpyAsync(c->d_sca_slot, slot.data(), c->nf, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaMemsetAsync(c->counters + CNT_SCAEV, 0, 8, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MCRT_OK;
}

int mcrt_scatter_events(mcrt_ctx *c, uint64_t *n_total_out, mcrt_scatter_event *events, uint64_t max_events, mcrt_mem where)
{
    if (!c || !n_total_out) return MCRT_EINVAL;
    if (!c->sca_ev) return fail(c, MCRT_ESTATE, "no scattering-event store: call mcrt_scatter_store first");
    unsigned long long n = 0ull;
    CUDA_TRY(c, cudaMemcpyAsync(&n, c->counters + CNT_SCAEV, 8, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    *n_total_out = n;
    if (events) {
        uint64_t m = n < c->sca_cap ? n : c->sca_cap;
        if (m > max_events) m = max_events;
        CUDA_TRY(c, cudaMemcpyAsync(events, c->sca_ev, m * sizeof(mcrt_scatter_event),
                                    where == MCRT_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    }
    return MCRT_OK;
}

int mcrt_ray_trace(mcrt_ctx *c, const mcrt_image_opts *io, double *F_emission, double *F_scatter, mcrt_mem where)
{
    if (!c || !io || !F_emission) return MCRT_EINVAL;
    if (!c->last_n || c->run.active) return fail(c, MCRT_ESTATE, "mcrt_ray_trace needs a finished run");
    if (c->mix || c->subR) return fail(c, MCRT_EINVAL, "mcrt_ray_trace: images of dust mixtures / divided grids are not defined");
    if (io->nx < 1 || io->ny < 1 || (size_t)io->nx * io->ny > ((size_t)1 << 28) || !(io->pixel_cm > 0.0) || !(io->distance_cm > 0.0) ||
        io->nu_bin < 0 || io->nu_bin >= c->nf)
        return fail(c, MCRT_EINVAL, "mcrt_ray_trace: bad image options");
    int rc;
    if ((rc = check_overflow(c))) return rc;
    RayParams R;
    {
        const double *z = io->e_z, *x = io->e_x;
        const double zn = sqrt(z[0] * z[0] + z[1] * z[1] + z[2] * z[2]);
        if (!(zn > 0.0)) return fail(c, MCRT_EINVAL, "e_z is zero");
        for (int a = 0; a < 3; ++a) R.ez[a] = z[a] / zn;
        const double dot = x[0] * R.ez[0] + x[1] * R.ez[1] + x[2] * R.ez[2];
        for (int a = 0; a < 3; ++a) R.ex[a] = x[a] - dot * R.ez[a];
        const double xn = sqrt(R.ex[0] * R.ex[0] + R.ex[1] * R.ex[1] + R.ex[2] * R.ex[2]);
        if (!(xn > 0.0)) return fail(c, MCRT_EINVAL, "e_x is parallel to e_z");
        for (int a = 0; a < 3; ++a) R.ex[a] /= xn;
        R.ey[0] = R.ez[1] * R.ex[2] - R.ez[2] * R.ex[1]; R.ey[1] = R.ez[2] * R.ex[0] - R.ez[0] * R.ex[2];
        R.ey[2] = R.ez[0] * R.ex[1] - R.ez[1] * R.ex[0];
    }
    const int j = io->nu_bin;
    R.inx = io->nx; R.iny = io->ny; R.pix_cells = io->pixel_cm / c->h;
    R.apix_d2 = io->pixel_cm * io->pixel_cm / (io->distance_cm * io->distance_cm);
    R.h = c->h; R.xi = c->xi; R.inv_fx = ldexp(1.0, -c->fx); R.cellfac = c->xi / (kFourPi * c->h * c->h * c->h);
    R.nu = c->nu[j]; R.inv_dnu = 1.0 / c->dnu[j];
    R.nx = c->nx; R.ny = c->ny; R.nz = c->nz; R.px = c->px; R.pxy = c->pxy; R.nT = c->nT; R.from_lucy = io->T_from_lucy; R.j = j; R.nf = c->nf;
    const size_t npix = (size_t)io->nx * io->ny;
    const size_t need = 2 * npix + (size_t)c->ns + 8;
    if (c->img_cap < need) {
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        if (c->img_buf) cudaFree(c->img_buf);
        c->img_buf = nullptr; c->img_cap = 0;
        if (cudaMalloc((void **)&c->img_buf, need * sizeof(double)) != cudaSuccess) return fail(c, MCRT_ENOMEM, "cudaMalloc of the image buffers failed");
        c->img_cap = need;
    }
    double *d_fe = (where == MCRT_DEVICE) ? F_emission : c->img_buf;
    double *d_fs = F_scatter ? ((where == MCRT_DEVICE) ? F_scatter : c->img_buf + npix) : nullptr;
    double *d_kabs = c->img_buf + 2 * npix;
    std::vector<double> kj(c->ns);
    for (int s = 0; s < c->ns; ++s) kj[s] = c->kabs[(size_t)s * c->nf + j];
    CUDA_TRY(c, cudaMemcpyAsync(d_kabs, kj.data(), c->ns * 8, cudaMemcpyHostToDevice, c->stream));
    // the sum over the stored events (Eq. 16), per cell, in the scratch array
    double *src = (double *)c->scratch;
    CUDA_TRY(c, cudaMemsetAsync(src, 0, c->nc * 8, c->stream));
    int slot = -1;
    for (size_t b = 0; b < c->sca_bins.size(); ++b) if (c->sca_bins[b] == j) slot = (int)b;
    if (c->sca_ev && slot >= 0 && F_scatter) {
        unsigned long long n = 0ull;
        CUDA_TRY(c, cudaMemcpyAsync(&n, c->counters + CNT_SCAEV, 8, cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        if (n > c->sca_cap) n = c->sca_cap;
        if (n) k_sca_source<<<stream_grid((size_t)n), 256, 0, c->stream>>>(c->sca_ev, n, slot, R.ez[0], R.ez[1], R.ez[2], c->cellw, c->d_g, c->nf, j,
                                                                         c->nx, c->ny, c->px, c->pxy, src);
    }
    k_ray_trace<<<(unsigned)((npix + 127) / 128), 128, 0, c->stream>>>(R, c->cellw, c->kabs_cnt, c->lfx, c->d_J, c->d_Tg, d_kabs, src, d_fe, d_fs);
    CUDA_TRY(c, cudaGetLastError());
    if (where == MCRT_HOST) {
        CUDA_TRY(c, cudaMemcpyAsync(F_emission, d_fe, npix * 8, cudaMemcpyDeviceToHost, c->stream));
        if (F_scatter) CUDA_TRY(c, cudaMemcpyAsync(F_scatter, d_fs, npix * 8, cudaMemcpyDeviceToHost, c->stream));
    }
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MCRT_OK;
}

int mcrt_read_tables(mcrt_ctx *c, double *dnu, double *J, double *cdf_B, double *cdf_dB, double *albedo, double *src_cdf)
{
    if (!c) return MCRT_EINVAL;
    if (!c->have_tables) return fail(c, MCRT_ESTATE, "tables not set");
    const size_t nsf = (size_t)c->ns * c->nf;
    // read back from the DEVICE copies: these are the values the kernels use
    if (dnu) CUDA_TRY(c, cudaMemcpyAsync(dnu, c->d_dnu, (size_t)c->nf * 8, cudaMemcpyDeviceToHost, c->stream));
    if (J) CUDA_TRY(c, cudaMemcpyAsync(J, c->d_J, (size_t)c->ns * c->nT * 8, cudaMemcpyDeviceToHost, c->stream));
    for (int pass = 0; pass < 2; ++pass) {
        double *dst = pass ? cdf_dB : cdf_B;
        if (!dst) continue;
        // the device rows are in Eytzinger order: read them back and put them in ascending order again
        const size_t rows = (size_t)c->ns * c->nT;
        std::vector<double> eyt(rows * c->nfs);
        CUDA_TRY(c, cudaMemcpyAsync(eyt.data(), pass ? c->d_cdfdB : c->d_cdfB, rows * c->nfs * 8, cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        for (size_t r = 0; r < rows; ++r)
            for (int k = 1; k <= c->nf; ++k) dst[r * c->nf + c->perm[k]] = eyt[r * c->nfs + k];
    }
    if (albedo) CUDA_TRY(c, cudaMemcpyAsync(albedo, c->d_albedo, nsf * 8, cudaMemcpyDeviceToHost, c->stream));
    if (src_cdf) {
        if (!c->have_source) return fail(c, MCRT_ESTATE, "source not set");
        CUDA_TRY(c, cudaMemcpyAsync(src_cdf, c->d_srccdf, (size_t)c->nf * 8, cudaMemcpyDeviceToHost, c->stream));
    }
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MCRT_OK;
}

int mcrt_philox_device(const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n)
{
    if (!ctr || !key || !out || n == 0) return MCRT_EINVAL;
    uint32_t *d = nullptr;
    if (cudaMalloc(&d, n * 10 * 4) != cudaSuccess) return fail(nullptr, MCRT_ENOMEM, "cudaMalloc failed");
    uint32_t *dc = d, *dk = d + 4 * n, *dout = d + 6 * n;
    cudaError_t e = cudaMemcpy(dc, ctr, n * 16, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dk, key, n * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_philox_test<<<(unsigned)((n + 255) / 256), 256>>>(dc, dk, dout, n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, dout, n * 16, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return fail(nullptr, MCRT_ECUDA, cudaGetErrorString(e));
    return MCRT_OK;
}

int mcrt_traj_math_device(const double *z, double *ln_z, double *sin_2piz, double *cos_2piz, uint64_t n)
{
    if (!z || !ln_z || !sin_2piz || !cos_2piz || n == 0) return MCRT_EINVAL;
    double *d = nullptr;
    if (cudaMalloc(&d, n * 4 * sizeof(double)) != cudaSuccess) return fail(nullptr, MCRT_ENOMEM, "cudaMalloc failed");
    std::vector<double> h(3 * n);
    cudaError_t e = cudaMemcpy(d, z, n * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_traj_math_test<<<(unsigned)((n + 255) / 256), 256>>>(d, d + n, n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(h.data(), d + n, 3 * n * sizeof(double), cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return fail(nullptr, MCRT_ECUDA, cudaGetErrorString(e));
    for (uint64_t i = 0; i < n; ++i) { ln_z[i] = h[3 * i]; sin_2piz[i] = h[3 * i + 1]; cos_2piz[i] = h[3 * i + 2]; }
    return MCRT_OK;
}

int mcrt_traj_math_device_static(const double *z, double *ln_z, double *sin_2piz, double *cos_2piz, uint64_t n)
{
    if (!z || !ln_z || !sin_2piz || !cos_2piz || n == 0) return MCRT_EINVAL;
    if (n > kStaticMaxN)
        return fail(nullptr, MCRT_EINVAL, "mcrt_traj_math_device_static: n exceeds MCRT_STATIC_MAX_N = " + std::to_string(kStaticMaxN) +
                                              " (the static device scratch holds no more; use mcrt_traj_math_device)");
    // The array's name is a host-side stand-in here: its device address comes from cudaGetSymbolAddress, once per
    // device, with that device current.
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, MCRT_ECUDA, cudaGetErrorString(e));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(nullptr, MCRT_EINVAL, "mcrt_traj_math_device_static: device ordinal out of range");
    double *d = g_static_scratch_ptr[dev].load(std::memory_order_acquire);
    if (!d) {
        e = cudaGetSymbolAddress((void **)&d, g_static_scratch);
        if (e != cudaSuccess || !d) return fail(nullptr, MCRT_ECUDA, std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e));
        g_static_scratch_ptr[dev].store(d, std::memory_order_release);
    }
    // layout: z | ln z | sin | cos, kStaticMaxN doubles each.  Nothing has to start at zero: every element read back
    // below is written by this call's copy or kernel; what an earlier call left beyond n is never read.
    e = cudaMemcpy(d, z, n * sizeof(double), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_traj_math_static<<<(unsigned)((n + 255) / 256), 256>>>(d, d + kStaticMaxN, d + 2 * kStaticMaxN, d + 3 * kStaticMaxN, n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(ln_z, d + kStaticMaxN, n * sizeof(double), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(sin_2piz, d + 2 * kStaticMaxN, n * sizeof(double), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(cos_2piz, d + 3 * kStaticMaxN, n * sizeof(double), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail(nullptr, MCRT_ECUDA, cudaGetErrorString(e));
    return MCRT_OK;
}

void mcrt_destroy(mcrt_ctx *c)
{
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    for (void *p : c->owned) cudaFree(p);
    for (int i = 0; i < 2; ++i) if (c->carry_buf[i]) cudaFree(c->carry_buf[i]);
    if (c->d_sca_slot) cudaFree(c->d_sca_slot);
    if (c->sca_ev) cudaFree(c->sca_ev);
    if (c->img_buf) cudaFree(c->img_buf);
    for (void *p : {(void *)c->d_mx_ncomp, (void *)c->d_mx_mat, (void *)c->d_mx_frac, (void *)c->d_mx_thr, (void *)c->d_kabs1_fx,
                    (void *)c->lfx1, (void *)c->kcnt1, (void *)c->kprev1, (void *)c->tidx1, (void *)c->d_kmax_diag, (void *)c->sub_cellw, (void *)c->sub_lfx, (void *)c->sub_kcnt, (void *)c->sub_kprev})
        if (p) cudaFree(p);
    delete c;
}

}  // extern "C"
