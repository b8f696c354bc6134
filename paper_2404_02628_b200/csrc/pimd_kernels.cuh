// CUDA kernels of the PIMD hot path (sm_100a, FP64, no tensor cores: d <= 3 is not a contraction).
// Notation follows arXiv 2404.02628 and DESIGN.md; 0-based indices in code.
//
// Exchange part in "generic recursion" form:
//   both Eq. 6 (forward) and Eq. 11 (backward) are instances of
//       R_i = log sum_{j<=i} sg_j exp( g_j - kk |rho_i - sig_j|^2 ),   g_{i+1} = R_i + cc_i,
//   kk = beta k_s / 2 = P/(2 beta), with
//   forward : rho_i = r_i^P, sig_j = r_j^1, g_j = a[j+1] = L_j + beta S[j] - (j+1) lambda
//   backward: rho_i = r_u^1, sig_j = r_l^P with u = N-1-i, l = N-1-j, g_j = q[l] - q[N]
//   cc = beta C(l,l+1) - lambda - ln(l+1)   (the same array, read in opposite order).
#pragma once
#include <cooperative_groups.h>
#include "pimd_math.cuh"

namespace pimd {

// ------------------------------------------------------------------------------------------
// small vector helpers; coordinate arrays are [n][D] packed doubles
// ------------------------------------------------------------------------------------------
template <int D> struct Vec { double v[D]; };

template <int D> PIMD_DEV Vec<D> ldvec(const double *p, size_t i)
{
    Vec<D> r;
    if constexpr (D == 2) {
        double2 t = *reinterpret_cast<const double2 *>(p + 2 * i);
        r.v[0] = t.x; r.v[1] = t.y;
    } else {
#pragma unroll
        for (int c = 0; c < D; ++c) r.v[c] = p[(size_t)D * i + c];
    }
    return r;
}
template <int D> PIMD_DEV void stvec(double *p, size_t i, const Vec<D> &a)
{
    if constexpr (D == 2) {
        *reinterpret_cast<double2 *>(p + 2 * i) = make_double2(a.v[0], a.v[1]);
    } else {
#pragma unroll
        for (int c = 0; c < D; ++c) p[(size_t)D * i + c] = a.v[c];
    }
}
template <int D> PIMD_DEV double dist2(const Vec<D> &a, const Vec<D> &b)
{
    double t = a.v[0] - b.v[0];
    double r2 = t * t;
#pragma unroll
    for (int c = 1; c < D; ++c) { t = a.v[c] - b.v[c]; r2 = fma(t, t, r2); }
    return r2;
}

PIMD_DEV int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
PIMD_DEV void st_release(int *p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
PIMD_DEV double2 ldcg2(const double2 *p) { return __ldcg(p); }
PIMD_DEV double ldcg1(const double *p) { return __ldcg(p); }
// A value that is its own "ready" flag: the consumer spins on the 8-byte word until it no longer holds this quiet-NaN
// payload (no arithmetic produces it); 8-byte accesses are single-copy atomic, so no fence and no second round trip.
constexpr unsigned long long PAN_EMPTY = 0x7ff8dead00c0ffeeull;
PIMD_DEV unsigned long long ld_relaxed_u64(const double *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
PIMD_DEV void st_relaxed_f64(double *p, double v)
{
    asm volatile("st.relaxed.gpu.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}

// Replica b of a batch lives `rs` bytes behind replica b-1 with the same layout: a kernel is handed the pointers of
// replica 0 and shifts them by blockIdx.{y,z} * rs.
template <class T> PIMD_DEV T *rshift(T *p, size_t off) { return (T *)((size_t)p + off); }

// status word bits (device -> host)
enum { ST_NONFINITE = 1, ST_NODE = 2 };

// ------------------------------------------------------------------------------------------
// Block-wide sum of one double per thread (deterministic order); result valid in thread 0.
// ------------------------------------------------------------------------------------------
template <int NT> PIMD_DEV double block_sum(double v, double *sh /* NT/32 doubles */)
{
    v = warp_sum(v);
    const int w = threadIdx.x >> 5, ln = threadIdx.x & 31;
    __syncthreads();
    if (ln == 0) sh[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = (ln < NT / 32) ? sh[ln] : 0.0;
        r = warp_sum(r);
    }
    return r;
}

// ==========================================================================================
// Step 1 of the hot path: spring + trap forces of every bead.
//   F[j][l] = intra-ring springs (Eq. 17; for j = 1, P the intra-ring half of
//             Eq. 15/16) - (1/P) omega^2 r (Eq. 4/19)
// grid (ceil(N/TB), P, B), block TB.  One thread owns one bead (j,l).  F is written (the pair kernel adds to it).
// EST: also accumulate U_trap and the radial histogram.
// ==========================================================================================
struct EstAccum {
    double utrap, upair, virpair, ec, pad[4];
};

template <int D, bool EST, int TB>
__global__ void __launch_bounds__(TB) k_bead(const double *__restrict__ x, double *__restrict__ F, int N, int P,
                                            double ks, double om2_over_P, EstAccum *est, double *hist, int nbins, double rmax,
                                            const double *__restrict__ halo_lo, const double *__restrict__ halo_hi, size_t rs)
{
    // P = number of bead slices held here.  A bead shard holds a contiguous range of the ring's slices and
    // gets the neighbouring ranks' boundary slices as halo_lo (the slice below local slice 0) / halo_hi (above local slice
    // P-1); NULL where the ring polymer itself ends (global bead 1 / bead P) and for an unsharded handle.
    __shared__ double red[TB / 32];
    const size_t off = (size_t)blockIdx.z * rs;
    x = rshift(x, off); F = rshift(F, off);
    const int j = blockIdx.y;
    const int l = blockIdx.x * TB + threadIdx.x;
    const bool valid = l < N;
    const double *xs = x + (size_t)j * N * D;
    Vec<D> r, f;
#pragma unroll
    for (int c = 0; c < D; ++c) { r.v[c] = 1e150; f.v[c] = 0.0; }
    double r2self = 0.0;
    if (valid) {
        r = ldvec<D>(xs, l);
        // ring-polymer springs inside particle l: neighbours j-1 and j+1 of the same particle.
        // Beads 1 and P get only their intra-ring neighbour here; the closing springs come from
        // the exchange kernels (Eq. 15, 16).
#pragma unroll
        for (int c = 0; c < D; ++c) f.v[c] = -om2_over_P * r.v[c];
        if (j > 0 || halo_lo != nullptr) {
            Vec<D> a = (j > 0) ? ldvec<D>(xs - (size_t)N * D, l) : ldvec<D>(rshift(halo_lo, off), l);
#pragma unroll
            for (int c = 0; c < D; ++c) f.v[c] -= ks * (r.v[c] - a.v[c]);
        }
        if (j < P - 1 || halo_hi != nullptr) {
            Vec<D> a = (j < P - 1) ? ldvec<D>(xs + (size_t)N * D, l) : ldvec<D>(rshift(halo_hi, off), l);
#pragma unroll
            for (int c = 0; c < D; ++c) f.v[c] -= ks * (r.v[c] - a.v[c]);
        }
#pragma unroll
        for (int c = 0; c < D; ++c) r2self = fma(r.v[c], r.v[c], r2self);
    }
    if (valid) stvec<D>(F + (size_t)j * N * D, l, f);
    if constexpr (EST) {
        est = rshift(est, off); hist = rshift(hist, off);
        double utr = valid ? 0.5 * om2_over_P * r2self : 0.0; // (1/P) 1/2 omega^2 r^2
        double s1 = block_sum<TB>(utr, red);
        if (threadIdx.x == 0) atomicAdd(&est->utrap, s1);
        if (nbins > 0 && valid) {
            const double rr = sqrt(r2self);
            if (rr < rmax) {
                int b = (int)(rr / rmax * nbins);
                if (b >= nbins) b = nbins - 1;
                atomicAdd(&hist[b], 1.0);
            }
        }
    }
}

// ==========================================================================================
// Step 3: closing springs the recursion needs outside the N x N part, E_int
// (Eq. 9), and the generic-recursion inputs.  One thread per particle.
// ==========================================================================================
struct ExchPtrs {
    double *rho[2], *sig[2], *cc[2];
    double2 *g[2];        // [N+1] gauge T_j (double-double): g_j = T_j + log|Zhat_j|
    double *gs[2];        // [N+1] Zhat_j: linear, signed, O(1)-ranged factor of exp(g_j)
    double2 *gprev[2];    // [N+1] g_j = T_j + log|Zhat_j| of the evaluation before the last one (gauge extrapolation)
    double *pan_m[2], *pan_s[2];
    int *cols_ready;      // [2]
    int *panel_ready[2];  // [NB]
    double *acc[2];       // [N][D+2]: sum w, sum w*sig (D), sum w*kk*r2
    double *pacc[2];      // [N][D+1]: the panel's share of sum w*sig (D) and sum w*kk*r2 per row, in the units of (pan_m, pan_s)
    double *eint, *cnext, *cself, *pnext;
    double *tpart;        // [2*nprepblocks] per-block partial sums of E_int, cnext
    double2 *rfin;        // [2]
    double *rsgn;         // [2]
    int *status;          // [2]: [0] ST_* bits of the current evaluation, [1] the same, sticky since pimd_set_state
};

// Per-replica parameters, kept in the replica's workspace region (a batch advances B replicas that differ in xi and
// in the noise seed with one set of launches).
struct RepParams {
    double xi, lambda /* ln|xi|, 0 for xi = 0 */, sx /* sgn xi */;
    unsigned long long seed;
};

PIMD_DEV ExchPtrs rshift(ExchPtrs p, size_t off)
{
    if (off == 0) return p;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        p.rho[k] = rshift(p.rho[k], off); p.sig[k] = rshift(p.sig[k], off); p.cc[k] = rshift(p.cc[k], off);
        p.g[k] = rshift(p.g[k], off); p.gs[k] = rshift(p.gs[k], off); p.gprev[k] = rshift(p.gprev[k], off);
        p.pan_m[k] = rshift(p.pan_m[k], off); p.pan_s[k] = rshift(p.pan_s[k], off);
        p.panel_ready[k] = rshift(p.panel_ready[k], off); p.acc[k] = rshift(p.acc[k], off); p.pacc[k] = rshift(p.pacc[k], off);
    }
    p.cols_ready = rshift(p.cols_ready, off);
    p.eint = rshift(p.eint, off); p.cnext = rshift(p.cnext, off); p.cself = rshift(p.cself, off); p.pnext = rshift(p.pnext, off);
    p.tpart = rshift(p.tpart, off); p.rfin = rshift(p.rfin, off); p.rsgn = rshift(p.rsgn, off); p.status = rshift(p.status, off);
    return p;
}

constexpr int PREP_SPLIT = 4; // thread groups that share the bead loop of a particle

// x: bead-major coordinates already offset to the first particle of this exchange problem (a species, SURVEY 8(f4),
// the recursion of Eq. 6 runs over that index range alone), `sl` doubles between consecutive bead slices,
// P slices; x1 / xP: the bead-1 and bead-P slices (same offset).  eint_in != NULL (bead shards): E_int comes
// summed over the ranks' slices instead of from the bead loop (x may be NULL).  grid (nprep, B).
template <int D, int TB>
__global__ void __launch_bounds__(TB *PREP_SPLIT) k_prep(const double *__restrict__ x, const double *__restrict__ x1s,
                                                        const double *__restrict__ xPs, const double *__restrict__ eint_in,
                                                        size_t sl, int N, int P, int NB, double ks, double kk, ExchPtrs p,
                                                        const RepParams *rp, int *gauge_misfit, int extrapolate, size_t rs)
{
    __shared__ double red[TB * PREP_SPLIT / 32];
    __shared__ double part_s[PREP_SPLIT][TB];
    const size_t off = (size_t)blockIdx.y * rs;
    p = rshift(p, off);
    x1s = rshift(x1s, off); xPs = rshift(xPs, off);
    const double lambda = rshift(rp, off)->lambda;
    const int lt = threadIdx.x % TB, part = threadIdx.x / TB;
    const int l = blockIdx.x * TB + lt;
    if (eint_in == nullptr) {
        // the P-1 bead differences of particle l, in PREP_SPLIT contiguous segments
        x = rshift(x, off);
        const int per = (P - 1 + PREP_SPLIT - 1) / PREP_SPLIT, j0 = 1 + part * per, j1 = min(P, j0 + per);
        double accp = 0.0;
        if (l < N && j0 < j1) {
            Vec<D> prev = ldvec<D>(x + (size_t)(j0 - 1) * sl, l);
            for (int j = j0; j < j1; ++j) {
                Vec<D> cur = ldvec<D>(x + (size_t)j * sl, l);
                accp += dist2<D>(cur, prev);
                prev = cur;
            }
        }
        part_s[part][lt] = accp;
    }
    __syncthreads();
    double e_int = 0.0, cn = 0.0;
    if (part == 0 && l < N) {
        if (eint_in == nullptr) {
            double acc = 0.0;
#pragma unroll
            for (int q = 0; q < PREP_SPLIT; ++q) acc += part_s[q][lt];
            e_int = 0.5 * ks * acc;
        } else {
            e_int = rshift(eint_in, off)[l];
        }
        const Vec<D> x1 = ldvec<D>(x1s, l);
        const Vec<D> xP = ldvec<D>(xPs, l);
        stvec<D>(p.rho[0], l, xP);
        stvec<D>(p.sig[0], l, x1);
        stvec<D>(p.rho[1], N - 1 - l, x1);
        stvec<D>(p.sig[1], N - 1 - l, xP);
        p.eint[l] = e_int;
        p.cself[l] = kk * dist2<D>(xP, x1);
        if (l < N - 1) {
            Vec<D> x1n = ldvec<D>(x1s, l + 1);
            cn = kk * dist2<D>(xP, x1n);
            const double c = cn - lambda - log((double)(l + 1));
            p.cc[0][l] = c;
            p.cc[1][N - 2 - l] = c;
        }
        p.cnext[l] = cn;
        if (l < NB) { p.panel_ready[0][l] = 0; p.panel_ready[1][l] = 0; }
#pragma unroll
        for (int dir = 0; dir < 2; ++dir) { // k_chain_spec reads the panel words as their own flags
            reinterpret_cast<unsigned long long *>(p.pan_m[dir])[l] = PAN_EMPTY;
            reinterpret_cast<unsigned long long *>(p.pan_s[dir])[l] = PAN_EMPTY;
        }
        // The gauge of the coming evaluation (k_chain_spec) from what the previous ones left behind: g_j = T_j + log|Zhat_j|
        // is the solution of the last evaluation; with `extrapolate` (two or more evaluations along one trajectory) its
        // change since the evaluation before is added once more.  A cloud that contracts or expands moves g by tens of
        // units per step, smoothly in time: the first-order prediction keeps the new solution within e^{O(1)} of the
        // gauge (measured: N = 40000 while the initial cloud falls into the trap, 48 rejected gauges in 120 steps -> see
        // profiles/r2_measurements.md).  Only a gauge: any value is correct, a bad one is caught by the acceptance band.
#pragma unroll
        for (int dir = 0; dir < 2; ++dir) {
            const double z = p.gs[dir][l + 1];
            const int ex = (__double2hiint(z) >> 20) & 0x7ff;
            if (ex != 0 && ex != 0x7ff) {
                const double2 gnow = dd_add_d(p.g[dir][l + 1], log(fabs(z)));
                double dlt = extrapolate ? dd_diff(gnow, p.gprev[dir][l + 1]) : 0.0;
                if (!(fabs(dlt) < 1e5)) dlt = 0.0;
                p.gprev[dir][l + 1] = gnow;
                p.g[dir][l + 1] = dd_add_d(gnow, dlt);
                p.gs[dir][l + 1] = z < 0.0 ? -1.0 : 1.0;
            }
        }
        if (l == 0) {
            p.g[0][0] = make_double2(-lambda, 0.0);
            p.g[1][0] = make_double2(0.0, 0.0);
            p.gs[0][0] = 1.0;
            p.gs[1][0] = 1.0;
            p.cols_ready[0] = 1;
            p.cols_ready[1] = 1;
            // status[0]: bits of the evaluation that starts here; status[1]: every bit seen since pimd_set_state
            p.status[1] |= p.status[0];
            p.status[0] = 0;
            if (blockIdx.y == 0) *gauge_misfit = 0;
        }
    }
    double s1 = block_sum<TB * PREP_SPLIT>(e_int, red);
    double s2 = block_sum<TB * PREP_SPLIT>(cn, red);
    if (threadIdx.x == 0) {
        p.tpart[2 * blockIdx.x] = s1;
        p.tpart[2 * blockIdx.x + 1] = s2;
    }
}

// ==========================================================================================
// Steps 4+5: the forward (Eq. 6) and backward (Eq. 11) recursions, blocked.
//
// grid (1 + nworkers, 2): blockIdx.y = direction, blockIdx.x == 0 the chain CTA, the others
// panel workers.  Rows/columns are cut into blocks of 32.  For row block K the LSE over columns
// j <= i is split into
//   old panel   j < 32 (K - LOOK)          -> a worker CTA, ahead of the chain (log-domain partial)
//   recent      32 (K - LOOK) <= j < 32 K  -> the chain CTA, all warps
//   diagonal    32 K <= j <= i             -> the chain CTA, sequential (the dependent part)
// The chain publishes (T_j, Zhat_j) with exp(g_j) = Zhat_j exp(T_j) and bumps cols_ready; workers
// publish (m, s) per row and set panel_ready[K].  All CTAs are co-resident (cooperative launch), so
// the spins terminate.
// ==========================================================================================
constexpr int CH_THREADS = 512;
constexpr int FP_TB = 128; // threads of a force-band / assembly task group (tail of the recursion kernels)
// doubles of shared memory one force-band task needs (a group of FP_TB = 128 threads)
template <int D> __host__ __device__ constexpr int fp_task_doubles() { return 2 * FP_TB + FP_TB + FP_TB * D + 4 * (D + 2) * (FP_TB / 4); }
constexpr int CH_WARPS = CH_THREADS / 32;
constexpr int CH_MAXLOOK = 3; // (4 L + 1) * 32 part entries are scaled by one pass of 512 threads

struct ChainArgs {
    int N, NB, look, nworkers;
    double kk;
    ExchPtrs p;                // replica 0; replica b of a batch is rs bytes further on (grid.z = replica)
    const RepParams *rp;       // likewise: sgn xi of the replica
    size_t rs;
    int look_fb;               // look-ahead of the max-plus recursion k_chain_spec falls back to (= look: the force band counts on it)
    double ks;                 // tail: spring constant, exterior-force outputs (replica 0, species offset applied), <E_c> partials
    double *Fex1, *FexP, *ecpart;
    int *gauge_misfit;         // k_chain_spec: one flag for the whole launch (all replicas fall back together)
    unsigned long long *fallbacks; // counts the launches that fell back
    unsigned long long *phase; // optional [16]: cycles of the forward chain CTA per phase (profiling), or NULL
};


// Shared-memory layout of the chain CTA (doubles); L = look.
template <int D> struct ChainSmem {
    int RB;                   // ring capacity in columns: 32 (L + 2)
    size_t ringT, ringZ, ringSig, rho, cc, dg, dgf, ue, ts, dlt, Gs, zeta, partM, partS, partG, apart, sh, total;
    __host__ __device__ explicit ChainSmem(int L)
    {
        RB = (L <= 2) ? 128 : 256;               // >= 32 (L + 2), a power of two
        size_t o = 0;
        ringT = o; o += 2 * (size_t)RB;          // double2 per column: the gauge T_j (double-double)
        ringZ = o; o += RB;                      // Zhat_j (signed)
        ringSig = o; o += (size_t)RB * D;
        rho = o; o += 2 * 32 * D;                // rows of blocks K, K+1 (double buffered)
        cc = o; o += 2 * 32;
        dg = o; o += 2 * 32 * 32;                // diagonal tiles of blocks K, K+1: tau, then M
        ue = o; o += 32 * 32;                    // exp part of block K's columns against the rows of block K+1
        dgf = o; o += 2 * 32 * 32 / 2;           // the same tau tiles as float (max-plus pass)
        ts = o; o += 20;                         // column gauges t_0..t_32 of the block (relative to Tref_K), float
        dlt = o; o += 40;                        // dlt[p] = t~_p - t_p (rounding remainder of the gauge)
        Gs = o; o += 32;                         // row gauges G_r
        zeta = o; o += 2 * 40;                   // Zhat of the block's columns, double buffered
        partM = o; o += 2 * (size_t)(4 * L + 1) * 32;    // contributions of earlier columns to the NEXT block's rows:
        partS = o; o += 2 * (size_t)(4 * L + 1) * 32; //   slot 0 panel (workers), then two half tiles per column block
        partG = o; o += (size_t)(4 * L + 1) * 32;    // float [2][(L+1)*32]: log|part| to within ln 2 (gauge start)
        apart = o; o += (size_t)(4 * L + 1) * 32;
        sh = o; o += 8;
        total = o;
    }
};

template <int D> size_t chain_smem_bytes_host(int look)
{
    const size_t chain = ChainSmem<D>(look).total * 8;
    const size_t worker = (size_t)CH_WARPS * 32 * (16 + 8 + D * 8) + (size_t)CH_WARPS * 32 * 16 + (size_t)CH_WARPS * 32 * 8 * (D + 1);
    const size_t tail = (size_t)(CH_THREADS / FP_TB) * fp_task_doubles<D>() * 8; // staging areas of exchange_tail
    const size_t m = chain > worker ? chain : worker;
    return m > tail ? m : tail;
}

PIMD_DEV void bar_sync_named(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }

// floor(log2|s|) * ln 2 from the exponent field: a lower bound of log|s| within ln 2 (gauge use only)
PIMD_DEV double approx_log_abs(double s)
{
    const int e = (__double2hiint(s) >> 20) & 0x7ff;
    return (double)(e - 1023) * 0.6931471805599453;
}

// ==========================================================================================
// The chain CTA.  Columns carry g_j = T_j + log|Zhat_j| as a
// double-double gauge T_j and a linear, signed, O(1)-ranged factor Zhat_j; no log or exp sits on
// the dependent path.  Per block K of 32 rows (rows and columns i0 = 32 K .. i0 + 31):
//   P1  warp 0: max-plus ("tropical") pass in FP32 -> column gauges t_p, row gauges G_r.  The io warp
//       publishes the previous block's columns to the workers and fetches their panel for block K+1.
//   P2  all: M[p][r] = exp(t~_p + tau[p][r] - G_r) <= 1;  Ahat parts = s exp(m - G_r); the exp part of
//       the contribution of block K's columns to the rows of block K+1 (T known, Zhat not yet), and the
//       complete contributions of the column blocks K+1-q, q = 2..L.
//   P3  warp 0: linear pass  acc_r = Ahat_r + sum_p M[p][r] Zhat_p,  Zhat_{r+1} = sx acc_r.
//   P4  all: finish block K's contribution (needs Zhat), publish T, Zhat to the ring, tau tile of
//       block K+1, coordinates of block K+2.
// Nothing but warp 0 (and a few global accesses of the io warp) runs during P1 and P3: shuffles share
// the SM's load/store pipe, and helper traffic placed beside the passes delayed them one for one.
// ==========================================================================================
template <int D, bool SGN>
__device__ void chain_cta(const ChainArgs &a, int dir, size_t roff, unsigned char *smem_raw, const double *etab)
{
    unsigned long long *const phase = (roff == 0) ? a.phase : nullptr;
    [[maybe_unused]] double sx = rshift(a.rp, roff)->sx; // this replica's sgn xi
    asm volatile("" : "+d"(sx));
    int N = a.N, L = a.look;
    // keep the two in registers: re-reading kernel parameters from the constant bank inside the block loop
    // was measured to stall the dependent warp for hundreds of cycles
    asm volatile("" : "+r"(N), "+r"(L));
    const ChainSmem<D> lay(L);
    const int RB = lay.RB;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    double *sm = reinterpret_cast<double *>(smem_raw);
    double2 *ring_T = reinterpret_cast<double2 *>(sm + lay.ringT);
    double *ring_Z = sm + lay.ringZ, *ring_sig = sm + lay.ringSig, *rho_s = sm + lay.rho, *cc_s = sm + lay.cc;
    float *dgf_s = reinterpret_cast<float *>(sm + lay.dgf), *ts_s = reinterpret_cast<float *>(sm + lay.ts);
    double *ue_s = sm + lay.ue;
    double *dg_s = sm + lay.dg, *dlt_s = sm + lay.dlt, *G_s = sm + lay.Gs, *zeta_s = sm + lay.zeta;
    float *part_g = reinterpret_cast<float *>(sm + lay.partG);
    double *part_m = sm + lay.partM, *part_s = sm + lay.partS, *apart_s = sm + lay.apart, *sh_s = sm + lay.sh;

    const double *rho = rshift(a.p.rho[dir], roff), *sig = rshift(a.p.sig[dir], roff), *cc = rshift(a.p.cc[dir], roff);
    double2 *g = rshift(a.p.g[dir], roff);
    double *gs = rshift(a.p.gs[dir], roff);
    const double kk = a.kk;
    const bool is_io = (warp == CH_WARPS - 1); // the warp that talks to global memory

    // coordinates and cc of block B -> shared (rows: rho_s[B&1], columns: ring_sig); zero padding
    auto load_block = [&](int B, int t, int nt) {
        for (int e = t; e < 32; e += nt) {
            const int i = B * 32 + e;
            Vec<D> pr, pc;
#pragma unroll
            for (int c = 0; c < D; ++c) { pr.v[c] = 0.0; pc.v[c] = 0.0; }
            double c0 = 0.0;
            if (i < N) {
                pr = ldvec<D>(rho, i);
                pc = ldvec<D>(sig, i);
                if (i < N - 1) c0 = cc[i];
            }
#pragma unroll
            for (int c = 0; c < D; ++c) {
                rho_s[((B & 1) * 32 + e) * D + c] = pr.v[c];
                ring_sig[(i & (RB - 1)) * D + c] = pc.v[c];
            }
            cc_s[(B & 1) * 32 + e] = c0;
        }
    };
    // diagonal tile of block B: dg[B&1][p][r] = -kk |rho_r - sig_{32B+p}|^2 for p <= r, -inf above
    auto diag_tile = [&](int B, int t, int nt) {
        double *dgB = dg_s + (B & 1) * 1024;
        for (int e = t; e < 1024; e += nt) {
            const int p = e >> 5, r = e & 31;
            const int slot = (B * 32 + p) & (RB - 1);
            Vec<D> pr, pc;
#pragma unroll
            for (int k = 0; k < D; ++k) { pr.v[k] = rho_s[((B & 1) * 32 + r) * D + k]; pc.v[k] = ring_sig[slot * D + k]; }
            const double tv = (p <= r) ? -kk * dist2<D>(pr, pc) : -INFINITY;
            dgB[e] = tv;
            dgf_s[(B & 1) * 1024 + e] = (float)tv;
        }
    };

    // ---- prologue: blocks 0 and 1, first column, empty parts
    load_block(0, tid, CH_THREADS);
    load_block(1, tid, CH_THREADS);
    if (tid == 0) {
        ring_T[0] = g[0];
        ring_Z[0] = 1.0;
        zeta_s[0] = 1.0;
        sh_s[0] = 0.0;
    }
    for (int e = tid; e < (4 * L + 1) * 32; e += CH_THREADS) { part_m[e] = -INFINITY; part_s[e] = 0.0; part_g[e] = -INFINITY; }
    __syncthreads();
    diag_tile(0, tid, CH_THREADS);
    __syncthreads();
    double2 pend_T = make_double2(0.0, 0.0); // io warp: columns computed in the previous block, to publish
    double pend_Z = 0.0;
    int pend_j = -1, pend_ready = 0;
    Vec<D> pre_rho, pre_sig; // io warp: coordinates of block K+2 in flight
    double pre_cc = 0.0;
    int panel_done = 0;      // io warp: the workers' panel of block K+1 has been fetched
    int bad = 0;             // warp 0: status bits of its rows
    double2 fin_T = make_double2(0.0, 0.0);
    double fin_G = 0.0, fin_acc = 1.0;
    const int NP = 4 * L + 1; // parts of the earlier-column sum of a row: panel, then four quarter tiles per block

    // Shuffles, shared-memory loads and stores all go through one pipe per SM (measured: 16 warps doing
    // warp reductions at once take ~4 cycles per shuffle).  The two dependent passes of warp 0 are chains of
    // shuffles, so whatever runs beside them must be register arithmetic with very few shared accesses:
    // tiles are computed with lane = row and a column loop (broadcast loads, no shuffles), two warps
    // per tile, each leaving a partial (max, sum) per row.

    // 8 columns [colbase, colbase+8) of a complete column block against row `pr`: partial log-domain sum
    auto part_tile = [&](const Vec<D> &pr, int colbase, const double2 &Tref_, float &mf, double &sv) {
        double t[8];
        mf = -INFINITY;
#pragma unroll
        for (int p = 0; p < 8; ++p) {
            const int slot = (colbase + p) & (RB - 1);
            Vec<D> pc;
#pragma unroll
            for (int c = 0; c < D; ++c) pc.v[c] = ring_sig[slot * D + c];
            t[p] = dd_diff(ring_T[slot], Tref_) - kk * dist2<D>(pr, pc);
            mf = fmaxf(mf, (float)t[p]);
        }
        const double m = (double)mf;
        double s0 = 0.0, s1 = 0.0;
#pragma unroll
        for (int p = 0; p < 8; p += 2) {
            s0 = fma(ring_Z[(colbase + p) & (RB - 1)], exp_tab(t[p] - m, etab), s0);
            s1 = fma(ring_Z[(colbase + p + 1) & (RB - 1)], exp_tab(t[p + 1] - m, etab), s1);
        }
        sv = s0 + s1;
    };

    // optional phase clock of the forward chain CTA: slot 2k-1 = warp 0's own time in phase k, slot 2k = its
    // wait at the barrier that ends phase k, slot 0 = loop overhead
    __shared__ long long ph_s[16];
    const bool tim = phase != nullptr && dir == 0 && tid == 0;
    if (tid < 16) ph_s[tid] = 0;
    long long tprev = clock64();
#define PH(k) do { if (tim) { const long long c__ = clock64(); ph_s[k] += c__ - tprev; tprev = c__; } } while (0)
    int NBk = a.NB;
    asm volatile("" : "+r"(NBk));
    for (int K = 0; K < NBk; ++K) {
        PH(0);
        const int i0 = K * 32, cur = K & 1, nxt = cur ^ 1;
        int nrows = min(32, N - i0);
        asm volatile("" : "+r"(nrows)); // no re-derivation from the constant bank later on
        const bool has_next = (K + 1 < NBk);
        const double2 Tref = ring_T[i0 & (RB - 1)];
        double *dgK = dg_s + cur * 1024;
        double *zK = zeta_s + cur * 40, *zN = zeta_s + nxt * 40;
        const double *pmK = part_m + cur * NP * 32, *psK = part_s + cur * NP * 32;
        double *pmN = part_m + nxt * NP * 32, *psN = part_s + nxt * NP * 32;
        const float *pgK = part_g + cur * NP * 32;
        float *pgN = part_g + nxt * NP * 32;
        double G = 0.0, accr = 0.0; // warp 0: row gauge and row sum of lane r
        float uMf = -INFINITY;

        // fetch the workers' panel of block K+1 (columns < 32 (K+1-L), relative to T_{32(K+1-L)})
        auto fetch_panel = [&](bool wait) {
            const int jrec0n = 32 * (K + 1 - L);
            double m = -INFINITY, s = 0.0;
            if (jrec0n > 0) {
                int ready = 0;
                if (lane == 0) {
                    ready = ld_acquire(&rshift(a.p.panel_ready[dir], roff)[K + 1]);
                    while (wait && ready == 0) ready = ld_acquire(&rshift(a.p.panel_ready[dir], roff)[K + 1]);
                }
                ready = __shfl_sync(0xffffffffu, ready, 0);
                if (!ready) return;
                const int i = i0 + 32 + lane;
                if (i < N) {
                    m = ldcg1(&rshift(a.p.pan_m[dir], roff)[i]) + dd_diff(ring_T[jrec0n & (RB - 1)], Tref);
                    s = ldcg1(&rshift(a.p.pan_s[dir], roff)[i]);
                }
            }
            pmN[lane] = m;
            psN[lane] = s;
            pgN[lane] = (float)(m + approx_log_abs(s));
            panel_done = 1;
        };

        // ================= P1: warp 0 max-plus pass.  Beside it: io warp publishes block K-1 and tries the
        // panel; warps 1, 2 the older column blocks against the rows of block K+1; warps 3..6 the tau
        // tile of block K+1
        if (warp == 0) {
            const int r = lane;
            const double my_cc = cc_s[cur * 32 + r];
            const double sh = sh_s[0];
            float mx = -INFINITY; // log of the earlier-column sum, to within ln 2 per part
            {
                float v[9];
#pragma unroll
                for (int k = 0; k < 9; ++k) v[k] = (k < NP) ? pgK[k * 32 + r] : -INFINITY;
                mx = fmaxf(fmaxf(fmaxf(fmaxf(v[0], v[1]), fmaxf(v[2], v[3])), fmaxf(fmaxf(v[4], v[5]), fmaxf(v[6], v[7]))), v[8]);
                for (int k = 9; k < NP; ++k) mx = fmaxf(mx, pgK[k * 32 + r]);
            }
            mx += (float)sh;
            // fully unrolled: a rolled loop costs ~20 more cycles per step (branch + divergence check)
            float tau[32];
#pragma unroll
            for (int p = 0; p < 32; ++p) tau[p] = dgf_s[cur * 1024 + p * 32 + lane];
            float tcur = 0.f, tmine = 0.f; // tmine: t_lane, kept in a register (no store inside the chain)
            const float ccf = (float)my_cc;
#pragma unroll
            for (int p = 0; p < 32; ++p) {
                mx = fmaxf(mx, tcur + tau[p]); // no effect once p > r
                tcur = __shfl_sync(0xffffffffu, mx + ccf, p);
                if (lane == p + 1) tmine = tcur;
            }
            G = (double)mx;
            const double tn = (double)(mx + ccf); // t_{r+1}, the value lane r broadcast at step r
            G_s[r] = G;
            dlt_s[r + 1] = (G - tn) + my_cc;      // t~_{r+1} - t_{r+1}, t~ = G + cc exactly
            ts_s[lane] = tmine;
            if (lane == 0) { ts_s[32] = tcur; dlt_s[0] = 0.0; }
        } else if (is_io) {
            if (pend_ready) {
                if (pend_j >= 0) { g[pend_j] = pend_T; gs[pend_j] = pend_Z; }
                // no fence: bar.warp.sync + st.release.gpu is cumulative over the other lanes' stores
                __syncwarp();
                if (lane == 0) st_release(&rshift(a.p.cols_ready, roff)[dir], min(N, i0 + 1));
                pend_ready = 0;
            }
            panel_done = 0;
            if (has_next) fetch_panel(false);
        } else if (has_next && warp <= 4) {
            Vec<D> pr;
#pragma unroll
            for (int c = 0; c < D; ++c) pr.v[c] = rho_s[(nxt * 32 + lane) * D + c];
            for (int q = 2; q <= L; ++q) {
                const int C = K + 1 - q, slotp = (4 * q - 4 + warp) * 32 + lane; // parts 5..8 for q = 2, ...
                float mf = -INFINITY;
                double sv = 0.0;
                if (C >= 0) part_tile(pr, C * 32 + (warp - 1) * 8, Tref, mf, sv);
                pmN[slotp] = (double)mf;
                psN[slotp] = sv;
                pgN[slotp] = mf + (float)approx_log_abs(sv);
            }
        } else if (has_next && warp <= 8) {
            // tau tile of block K+1, lane = row, 8 columns per warp
            double *dgB = dg_s + nxt * 1024;
            Vec<D> pr;
#pragma unroll
            for (int c = 0; c < D; ++c) pr.v[c] = rho_s[(nxt * 32 + lane) * D + c];
#pragma unroll
            for (int pp = 0; pp < 8; ++pp) {
                const int p = (warp - 5) * 8 + pp;
                Vec<D> pc;
#pragma unroll
                for (int c = 0; c < D; ++c) pc.v[c] = ring_sig[((i0 + 32 + p) & (RB - 1)) * D + c];
                const double tv = (p <= lane) ? -kk * dist2<D>(pr, pc) : -INFINITY;
                dgB[p * 32 + lane] = tv;
                dgf_s[nxt * 1024 + p * 32 + lane] = (float)tv;
            }
        }
        PH(1);
        __syncthreads();
        PH(2);

        // ================= P2 (all threads): M pass and the earlier-column parts under the row gauges
        {
            // two independent exps per thread; tau = -inf above the diagonal gives exactly 0
            const int r = tid & 31, p0 = tid >> 5, p1 = p0 + 16;
            const double Gr = G_s[r];
            const double a0 = (((double)ts_s[p0] - Gr) + dgK[tid]) + dlt_s[p0];
            const double a1 = (((double)ts_s[p1] - Gr) + dgK[tid + 512]) + dlt_s[p1];
            double m0 = exp_tab(a0, etab), m1 = exp_tab(a1, etab);
            if constexpr (SGN) { if (p0 >= 1) m0 *= sx; m1 *= sx; }
            dgK[tid] = m0;
            dgK[tid + 512] = m1;
            const int ai = tid - (CH_THREADS - NP * 32); // the last warps also scale the earlier-column parts
            if (ai >= 0) apart_s[ai] = psK[ai] * exp_tab((pmK[ai] + sh_s[0]) - G_s[ai & 31], etab);
        }
        PH(3);
        __syncthreads();
        PH(4);

        // ================= P3: warp 0 linear pass.  Beside it: io warp (panel if not ready in P1, loads of
        // block K+2's coordinates); warps 1, 2 the exp part of block K's columns against the rows of block K+1
        if (warp == 0) {
            double M[32];
#pragma unroll
            for (int p = 0; p < 32; ++p) M[p] = dgK[p * 32 + lane];
            double acc = 0.0;
            {
                double v[9]; // independent loads first (a runtime-count loop serialises on the load latency)
#pragma unroll
                for (int k = 0; k < 9; ++k) v[k] = (k < NP) ? apart_s[k * 32 + lane] : 0.0;
                acc = (((v[0] + v[1]) + (v[2] + v[3])) + ((v[4] + v[5]) + (v[6] + v[7]))) + v[8];
                for (int k = 9; k < NP; ++k) acc += apart_s[k * 32 + lane];
            }
            double zc = zK[0], zmine = zc; // zmine: X^_{lane-1}, kept in a register
#pragma unroll
            for (int p = 0; p < 32; ++p) {
                acc = fma(M[p], zc, acc);  // M[p][r] = 0 once p > r
                zc = shfl_bcast(acc, p);   // X^_p; Zhat_{p+1} = sx X^_p (sx is folded into M)
                if (lane == p + 1) zmine = zc;
            }
            accr = acc;
            if (lane >= 1) zK[lane] = SGN ? sx * zmine : zmine;
            if (lane == 0) { zK[32] = SGN ? sx * zc : zc; zN[0] = SGN ? sx * zc : zc; }
        } else if (is_io) {
            if (has_next) {
                if (!panel_done) fetch_panel(true);
                const int i = i0 + 64 + lane;
#pragma unroll
                for (int c = 0; c < D; ++c) { pre_rho.v[c] = 0.0; pre_sig.v[c] = 0.0; }
                pre_cc = 0.0;
                if (i < N) {
                    pre_rho = ldvec<D>(rho, i);
                    pre_sig = ldvec<D>(sig, i);
                    if (i < N - 1) pre_cc = cc[i];
                }
            }
        } else if (has_next && warp <= 4) {
            Vec<D> pr;
#pragma unroll
            for (int c = 0; c < D; ++c) pr.v[c] = rho_s[(nxt * 32 + lane) * D + c];
            const int c0 = (warp - 1) * 8;
            double u[8];
#pragma unroll
            for (int p = 0; p < 8; ++p) {
                Vec<D> pc;
#pragma unroll
                for (int c = 0; c < D; ++c) pc.v[c] = ring_sig[((i0 + c0 + p) & (RB - 1)) * D + c];
                u[p] = ((double)ts_s[c0 + p] - kk * dist2<D>(pr, pc)) + dlt_s[c0 + p];
                uMf = fmaxf(uMf, (float)u[p]);
            }
            const double m = (double)uMf;
#pragma unroll
            for (int p = 0; p < 8; ++p) ue_s[(c0 + p) * 32 + lane] = exp_tab(u[p] - m, etab);
        }
        PH(5);
        __syncthreads();
        PH(6);

        // ================= P4: warps 1, 2 finish block K's contribution (needs Zhat); warp 0 publishes T and
        // Zhat to the ring; io warp takes its copy for the workers and stores block K+2's coordinates
        if (warp == 0) {
            if (lane < nrows) { // status and the final row are dealt with once, after the loop
                if (accr == 0.0) bad |= ST_NODE;
                else if (!(fabs(accr) < INFINITY)) bad |= ST_NONFINITE;
            }
            if (!has_next) { fin_T = Tref; fin_G = G; fin_acc = accr; }
        } else if (warp == 9) {
            // T and Zhat of the columns this block produced -> ring
            const int jn = i0 + lane + 1;
            if (jn < N) {
                ring_T[jn & (RB - 1)] = dd_add_d(dd_add_d(Tref, (double)ts_s[lane + 1]), dlt_s[lane + 1]);
                ring_Z[jn & (RB - 1)] = zK[lane + 1];
            }
            if (lane == 0) sh_s[0] = -((double)ts_s[32] + dlt_s[32]);
        } else if (is_io) {
            const int jn = i0 + lane + 1;
            pend_j = (jn <= N) ? jn : -1; // column N too: its T is the last row's gauge for k_chain_spec
            pend_T = dd_add_d(dd_add_d(Tref, (double)ts_s[lane + 1]), dlt_s[lane + 1]);
            pend_Z = zK[lane + 1];
            pend_ready = 1;
            if (has_next) { // block K+2 (zeros beyond N): free buffers, first read in P1 of block K+1
#pragma unroll
                for (int c = 0; c < D; ++c) {
                    rho_s[(cur * 32 + lane) * D + c] = pre_rho.v[c];
                    ring_sig[((i0 + 64 + lane) & (RB - 1)) * D + c] = pre_sig.v[c];
                }
                cc_s[cur * 32 + lane] = pre_cc;
            }
        } else if (has_next && warp <= 4) {
            const int c0 = (warp - 1) * 8;
            double s0 = 0.0, s1 = 0.0;
#pragma unroll
            for (int p = 0; p < 8; p += 2) {
                s0 = fma(ue_s[(c0 + p) * 32 + lane], zK[c0 + p], s0);
                s1 = fma(ue_s[(c0 + p + 1) * 32 + lane], zK[c0 + p + 1], s1);
            }
            const double sv = s0 + s1, m = (double)uMf;
            pmN[warp * 32 + lane] = m; // parts 1..4
            psN[warp * 32 + lane] = sv;
            pgN[warp * 32 + lane] = (float)(m + approx_log_abs(sv));
        }
        PH(7);
        __syncthreads();
        PH(8);
    }
#undef PH
    if (tim) {
        for (int k = 0; k < 16; ++k) phase[k] += (unsigned long long)ph_s[k];
    }
    if (warp == 0) {
        // R_{N-1} = T + G + log|X^| of the last row, its sign, and the status of all rows
        if (lane == (N - 1) % 32) {
            rshift(a.p.rfin, roff)[dir] = dd_add_d(dd_add_d(fin_T, fin_G), log(fabs(fin_acc)));
            rshift(a.p.rsgn, roff)[dir] = (fin_acc < 0.0) ? -1.0 : 1.0;
        }
        if (bad) atomicOr(rshift(a.p.status, roff), bad);
    }
    if (is_io && pend_ready) {
        if (pend_j >= 0) { g[pend_j] = pend_T; gs[pend_j] = pend_Z; }
        // no fence: bar.warp.sync + st.release.gpu is cumulative over the other lanes' stores
        __syncwarp();
        if (lane == 0) st_release(&rshift(a.p.cols_ready, roff)[dir], N);
    }
}

// ==========================================================================================
// The chain CTA with a STALE GAUGE.  Between two MD steps the
// solution moves by a factor e^{O(1)} per column, so the gauge T_j the previous evaluation left in
// g[dir] (refreshed by k_prep so that |Zhat| is in [1,2)) is as good as a fresh max-plus pass: with it
// the column gauges t_p, the row gauges G_r = t_{r+1} - cc_r, the tile M = exp(t_p + tau - G_r), the
// scaled contributions of all earlier columns and even the NEW T_j are known before the block is
// reached.  What remains dependent is one linear pass per 32-row block (DFMA + SHFL per row), and
// everything it needs is prepared by the other warps one or two blocks ahead:
//   window K (while warp 0 solves block K):
//     warp 15   publishes block K-1 (T, Zhat) to the workers, prefetches coordinates / cc / old T of block K+3
//     warp 14   fetches and scales the workers' panel of block K+1
//     warp 1    gauges of block K+2 (and the new T of its columns -> ring)
//     warps 2-9   M tile of block K+1
//     warps 10-13 contributions of the column blocks K+1-q, q = 2..L, to the rows of block K+1
//     then warps 1-13: E'(K+2) = exp part of block K+1's columns against the rows of block K+2
//   At the end of a block the exponent of Zhat of its last column is taken out of the following blocks'
//   frame (exact powers of two), so a systematic drift of the solution along the chain cannot overflow.
//   warp 0 folds E'(K+1) Zhat into the next block's start value inside its own loop (one more DFMA per
//   step, off the dependent path), so one block-wide barrier per block is all the synchronisation.
// A row sum outside 2^+-64 of its gauge (the gauge no longer fits: state replaced, a jump) raises the misfit flag;
// k_chain_spec then redoes the recursion with the max-plus code after a grid barrier.
// ==========================================================================================
#ifndef PIMD_SPEC_NHW
#define PIMD_SPEC_NHW 9
#endif
constexpr int SPEC_NHW = PIMD_SPEC_NHW;                     // helper warps of the stale-gauge chain CTA: 9 or 12
constexpr int SPEC_NCOL = (32 + SPEC_NHW - 1) / SPEC_NHW;  // columns of a tile per helper warp
#ifndef PIMD_FACT_LIMIT
#define PIMD_FACT_LIMIT 1024.0
#endif
// doubles per column entry of the helpers' tables: A_p, sigma'_p[D], t_p, dl_p, padded to an even count (LDS.128 reads)
__host__ __device__ constexpr int SPEC_CW(int D) { return (3 + D + 1) / 2 * 2; }
constexpr double SKIP_BELOW = -260.0;           // helper batches whose entries all lie below e^SKIP_BELOW of the row's gauge are dropped
constexpr double FACT_LIMIT = PIMD_FACT_LIMIT; // largest tabulated term for which the factorised exponent arguments are used

template <int D> struct SpecSmem {
    int RB;
    size_t ringT, ringZ, ringSig, rho, cc, traw, colT, Gs, trefn, mt, ue, baseT, baseP, zmail, kacc, fmode, ctab, rtab, total;
    __host__ __device__ SpecSmem()
    {
        RB = 256;
        size_t o = 0;
        ringT = o; o += 2 * (size_t)RB;
        ringZ = o; o += RB;
        ringSig = o; o += (size_t)RB * D;
        rho = o; o += 8 * 32 * D;     // rows of blocks B & 7
        cc = o; o += 8 * 32;
        traw = o; o += 8 * 2 * 34;    // old T (double-double) of columns 32B .. 32B+32
        colT = o; o += 8 * 2 * 34;    // column gauges of block B & 7: (t_p as float value, remainder), p = 0..32
        Gs = o; o += 8 * 32;
        trefn = o; o += 8 * 2;        // new T of column 32B (double-double)
        mt = o; o += 2 * 1024;        // M tiles of blocks B & 1
        ue = o; o += 2 * 1024;        // E'(B & 1)
        baseT = o; o += 2 * 2 * SPEC_NHW * 32; // [B & 1][q - 2][helper warp][row] partial sums of the older column blocks
        baseP = o; o += 2 * 32;       // scaled panel for block B & 1
        zmail = o; o += 2 * 32;       // Zhat of the columns block B & 1 produced, for the io warp
        kacc = o; o += 4;             // int[8]: power of two taken out of Zhat up to the start of block B & 7
        fmode = o; o += 2;            // int[2] (two doubles: what follows stays 16-byte aligned): the tables of window & 1 hold the factorised terms (1) or the plain pieces (0)
        ctab = o; o += 2 * 4 * 32 * SPEC_CW(D); // [window & 1][set][column]: (A_p, sigma'_p, t_p, dl_p) padded to whole double2, see col_row_terms
        rtab = o; o += 2 * 2 * 32 * (2 + 2 * D); // [window & 1][set][row]: (B_r, 2 kk rho'_r, G_r, rho'_r)
        total = o;
    }
};

template <int D, bool SGN>
__device__ void chain_cta_spec(const ChainArgs &a, int dir, size_t roff, unsigned char *smem_raw, const double *etab64)
{
    unsigned long long *const phase = (roff == 0) ? a.phase : nullptr;
    [[maybe_unused]] double sx = rshift(a.rp, roff)->sx; // this replica's sgn xi
    asm volatile("" : "+d"(sx));
    int N = a.N, L = a.look, NBk = a.NB;
    asm volatile("" : "+r"(N), "+r"(L), "+r"(NBk));
    const SpecSmem<D> lay;
    __shared__ long long ph_s[16]; // phase clock (profiling)
    constexpr int RB = 256;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    double *sm = reinterpret_cast<double *>(smem_raw);
    double2 *ring_T = reinterpret_cast<double2 *>(sm + lay.ringT);
    double *ring_Z = sm + lay.ringZ, *ring_sig = sm + lay.ringSig, *rho_s = sm + lay.rho, *cc_s = sm + lay.cc;
    double2 *traw_s = reinterpret_cast<double2 *>(sm + lay.traw);
    double2 *colT_s = reinterpret_cast<double2 *>(sm + lay.colT);
    double *G_s = sm + lay.Gs;
    double2 *trefn_s = reinterpret_cast<double2 *>(sm + lay.trefn);
    double *mt_s = sm + lay.mt, *ue_s = sm + lay.ue, *baseT_s = sm + lay.baseT, *baseP_s = sm + lay.baseP, *zmail_s = sm + lay.zmail;
    int *kacc_s = reinterpret_cast<int *>(sm + lay.kacc);
    double *ctab_s = sm + lay.ctab, *rtab_s = sm + lay.rtab;
    int *fmode_s = reinterpret_cast<int *>(sm + lay.fmode);

    const double *rho = rshift(a.p.rho[dir], roff), *sig = rshift(a.p.sig[dir], roff), *cc = rshift(a.p.cc[dir], roff);
    double2 *g = rshift(a.p.g[dir], roff);
    double *gs = rshift(a.p.gs[dir], roff);
    const double kk = a.kk;

    // ---- pieces of the preparation, written for a group of `nt` threads with index `t`
    // coordinates, cc and the old gauge of block B -> shared (32 threads are enough); zeros beyond N
    auto load_raw = [&](int B, int t, int nt) {
        const int b3 = B & 7;
        for (int e = t; e < 33; e += nt) {
            const int i = B * 32 + e;
            // beyond the last column the gauge continues flat: padded rows must stay finite (0 * inf = NaN would
            // leak into the real rows through their zero matrix entries)
            const double2 told = ldcg2(&g[min(i, N)]);
            traw_s[b3 * 34 + e] = told;
            if (e < 32) {
                Vec<D> pr, pc;
#pragma unroll
                for (int c = 0; c < D; ++c) { pr.v[c] = 0.0; pc.v[c] = 0.0; }
                double c0 = 0.0;
                if (i < N) {
                    pr = ldvec<D>(rho, i);
                    pc = ldvec<D>(sig, i);
                    if (i < N - 1) c0 = cc[i];
                }
#pragma unroll
                for (int c = 0; c < D; ++c) {
                    rho_s[(b3 * 32 + e) * D + c] = pr.v[c];
                    ring_sig[(i & (RB - 1)) * D + c] = pc.v[c];
                }
                cc_s[b3 * 32 + e] = c0;
            }
        }
    };
    // gauges of block B (one warp, lane = row r): t_{r+1} from the old T, G_r = t_{r+1} - cc_r, the new
    // gauge t~_{r+1} = G_r + cc_r exactly (float t + remainder dlt, kept as one double2 per column), the new T of
    // column 32B+r+1
    auto gauges = [&](int B) {
        const int b7 = B & 7, r = lane;
        const double told = dd_diff(traw_s[b7 * 34 + r + 1], traw_s[b7 * 34]);
        const double my_cc = cc_s[b7 * 32 + r];
        const float Gf = (float)(told - my_cc);
        const float tn = Gf + (float)my_cc;
        const double dl = ((double)Gf - (double)tn) + my_cc;
        G_s[b7 * 32 + r] = (double)Gf;
        colT_s[b7 * 34 + r + 1] = make_double2((double)tn, dl);
        if (r == 0) colT_s[b7 * 34] = make_double2(0.0, 0.0);
        const double2 Tn = dd_add_d(dd_add_d(trefn_s[b7], (double)tn), dl);
        ring_T[(B * 32 + r + 1) & (RB - 1)] = Tn;
        if (r == 31) trefn_s[(B + 1) & 7] = Tn;
    };
    // What the helper warps prepare during window K, lane = row throughout (row data in registers, column data by
    // broadcast loads, no shuffles), helper warp hw of 9 takes columns hw, hw+9, hw+18, hw+27 of every tile as one
    // batch: four exponent arguments first, then four exponentials, then the stores:
    //   M(B)[p][r]  = exp(t~_p + tau[p][r] - G_r), p <= r, sx folded in for p >= 1              (B = K+1)
    //   base(B)     = sum over the columns of block B-q (q = 2..L) of Zhat exp(T - T_ref(B) + tau - G_r), one
    //                 partial sum per (q, helper warp, row), in the frame of block B-q              (B = K+1)
    //   E'(B)[p][r] = column p of block B-1 against row r of block B, relative to the new T of column 32B,
    //                 scaled by exp(-G_r(B)), everything but the factor Zhat_p, sx folded in for p >= 1 (B = K+2)
    // Exponent arguments in three FP64 instructions per entry.  With an origin o (row 0 of the row block, so that every
    // term stays of the size of the distances themselves) and rho' = rho_r - o, sigma' = sigma_p - o,
    //     (column term) - G_r - kk |rho_r - sigma_p|^2 = A_p + B_r + sum_c (2 kk rho'_c) sigma'_c,
    //     A_p = (column term) - kk |sigma'_p|^2,   B_r = -G_r - kk |rho'_r|^2.
    // One warp tabulates, during window K, what the helpers use during window K+1 (lane = column / row):
    //   rows    set 0: block K+2 (M and base of block K+2),          set 1: block K+3 (E'(K+3))
    //   columns set 0: block K+2 for M(K+2), origin o(K+2)            set 1: block K+2 for E'(K+3), origin o(K+3)
    //           set 2, 3: blocks K, K-1 for base(K+2), origin o(K+2)
    // The factorised form costs 1 + D instructions per entry but cancels numbers of the size kk R^2 + |gauge| (R = extent of
    // the blocks about the origin): its rounding error, a few ulp of that size, is common to a row or a column of a tile
    // and travels down the chain with Zhat.  It is used only while every tabulated term stays below FACT_LIMIT (a
    // thermalised cloud: kk R^2 ~ 10^1..10^2); otherwise -- the spread-out initial clouds of the BASELINE configurations,
    // kk R^2 ~ 10^4 -- the window's tables hold the plain pieces and the entries are formed the direct way,
    //     ((t_p - G_r) + dl_p) - kk |rho'_r - sigma'_p|^2,   t_p, G_r float-valued so that their difference is exact,
    // 3 + 2 D instructions with the accuracy of the max-plus kernel (measured: forces 1.4e-9 -> see profiles/r2_measurements.md).
    auto col_row_terms = [&](int K) {
        constexpr int W = 2 + 2 * D, CW = SPEC_CW(D);
        double *cA = ctab_s + (K & 1) * (4 * 32 * CW), *rA = rtab_s + (K & 1) * (2 * 32 * W);
        const int B2 = K + 2, B3 = K + 3, b2 = B2 & 7, b3 = B3 & 7;
        Vec<D> o2, o3;
#pragma unroll
        for (int c = 0; c < D; ++c) { o2.v[c] = rho_s[(b2 * 32) * D + c]; o3.v[c] = rho_s[(b3 * 32) * D + c]; }
        double rG[2], rn2[2], rp_[2][D];
        bool big = false;
#pragma unroll
        for (int set = 0; set < 2; ++set) {
            const int b = set ? b3 : b2;
            rn2[set] = 0.0;
#pragma unroll
            for (int c = 0; c < D; ++c) {
                rp_[set][c] = rho_s[(b * 32 + lane) * D + c] - (set ? o3.v[c] : o2.v[c]);
                rn2[set] = fma(rp_[set][c], rp_[set][c], rn2[set]);
            }
            rG[set] = G_s[b * 32 + lane];
            big = big || !(kk * rn2[set] + fabs(rG[set]) < FACT_LIMIT);
        }
        const double2 ct = colT_s[b2 * 34 + lane], c32 = colT_s[b2 * 34 + 32], Tref2 = trefn_s[b2];
        double th[4], tl[4], cn2[4], sp_[4][D];
#pragma unroll
        for (int set = 0; set < 4; ++set) {
            const int C = (set < 2) ? B2 : B2 - set; // column block
            const int slot = (max(C, 0) * 32 + lane) & (RB - 1);
            if (set == 0) { th[set] = ct.x; tl[set] = ct.y; }
            else if (set == 1) { th[set] = ct.x - c32.x; tl[set] = ct.y - c32.y; } // float-valued parts: exact
            else {
                const double2 Tp = ring_T[slot];
                th[set] = dd_diff(Tp, Tref2);
                tl[set] = ((Tp.x - Tref2.x) - th[set]) + (Tp.y - Tref2.y); // what the rounding of th dropped
            }
            cn2[set] = 0.0;
#pragma unroll
            for (int c = 0; c < D; ++c) {
                sp_[set][c] = ring_sig[slot * D + c] - (set == 1 ? o3.v[c] : o2.v[c]);
                cn2[set] = fma(sp_[set][c], sp_[set][c], cn2[set]);
            }
            if (C >= 0) big = big || !(kk * cn2[set] + fabs(th[set]) < FACT_LIMIT);
        }
        const bool fact = __any_sync(0xffffffffu, big) == 0;
        if (lane == 0) {
            fmode_s[K & 1] = fact ? 1 : 0;
            if (phase != nullptr && dir == 0 && fact && K >= 0) ph_s[6] += 1; // profiling: windows with factorised arguments
        }
#pragma unroll
        for (int set = 0; set < 2; ++set) {
            double *r_ = rA + (set * 32 + lane) * W;
            r_[0] = fma(-kk, rn2[set], -rG[set]);
            r_[1 + D] = rG[set];
#pragma unroll
            for (int c = 0; c < D; ++c) { r_[1 + c] = 2.0 * kk * rp_[set][c]; r_[2 + D + c] = rp_[set][c]; }
        }
#pragma unroll
        for (int set = 0; set < 4; ++set) {
            const int C = (set < 2) ? B2 : B2 - set;
            if (C < 0) continue;
            double *c_ = cA + (set * 32 + lane) * CW;
#pragma unroll
            for (int c = 0; c < D; ++c) c_[1 + c] = sp_[set][c];
            c_[0] = fma(-kk, cn2[set], th[set] + tl[set]);
            c_[1 + D] = th[set];
            c_[2 + D] = tl[set];
        }
    };
    // one entry's exponent argument from the column's and the row's table entries (cp, rp):
    // factorised, A_p + B_r + sum_c w_c sigma'_c -- final in a `fact` window, else good to ~1e-11, enough to tell a dead batch
    // Table entries are read as double2 (LDS.128): the helpers' shared-memory instructions, not their arithmetic, set
    // the block time (the SM has one pipe for LDS, STS and the dependent warp's shuffles).
    auto ld_entry = [&](const double *q, double *v, int nd2) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (k < nd2) { const double2 t = *reinterpret_cast<const double2 *>(q + 2 * k); v[2 * k] = t.x; v[2 * k + 1] = t.y; }
        }
    };
    auto entry_arg = [&](const double *cp, const double *rp) {
        double c[8];
        ld_entry(cp, c, (D + 2) / 2); // A_p, sigma'_p
        double t = c[0] + rp[0];
#pragma unroll
        for (int k = 0; k < D; ++k) t = fma(rp[1 + k], c[1 + k], t);
        return t;
    };
    // direct, ((t_p - G_r) + dl_p) - kk |rho'_r - sigma'_p|^2
    auto entry_arg_direct = [&](const double *cp, const double *rp) {
        double c[8];
        ld_entry(cp, c, (D + 4) / 2); // sigma'_p, t_p, dl_p
        double dd = rp[2 + D] - c[1];
        double r2 = dd * dd;
#pragma unroll
        for (int k = 1; k < D; ++k) { dd = rp[2 + D + k] - c[1 + k]; r2 = fma(dd, dd, r2); }
        return fma(-kk, r2, (c[1 + D] - rp[1 + D]) + c[2 + D]);
    };
    auto batch_is_live = [&](const double *arg) {
        bool live = false;
#pragma unroll
        for (int k = 0; k < SPEC_NCOL; ++k) live = live || !(arg[k] < SKIP_BELOW - 1.0); // NaN counts as live; the margin covers the factorised form's error
        return __any_sync(0xffffffffu, live) != 0;
    };
    auto helper_tasks = [&](int K, int hw) {
        constexpr int CW = SPEC_CW(D), RW = 2 + 2 * D;
        const bool fact = fmode_s[(K + 1) & 1] != 0; // mode of the tables this window reads (warp-uniform)
        const bool tht = phase != nullptr && dir == 0 && lane == 0 && hw == 0;
        const long long ht0 = clock64();
        {   // ---- M(K+1): only p <= r is needed, so columns pp and 31-pp share one pass of 32 lanes (33 entries; the
            // odd one, row 31 of column 31-pp, goes to a 17th pass); above the diagonal the tile stays 0 from the start.
            // Helper warp hw takes passes hw and hw + 9.
            const int B = K + 1;
            double *mB = mt_s + (B & 1) * 1024;
            const double *cA = ctab_s + ((K + 1) & 1) * (4 * 32 * CW), *rA = rtab_s + ((K + 1) & 1) * (2 * 32 * RW);
            double arg[2];
            int idx[2];
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const int pass = hw + SPEC_NHW * k;
                int p, r;
                if (pass < 16) {
                    if (lane >= pass) { p = pass; r = lane; } else { p = 31 - pass; r = 31 - pass + lane; }
                } else {
                    p = 31 - (lane & 15); r = 31; // 16 leftovers (each written twice, same value)
                }
                double rr[8];
                ld_entry(rA + r * RW, rr, fact ? (D + 2) / 2 : (2 + 2 * D) / 2);
                arg[k] = fact ? entry_arg(cA + p * CW, rr) : entry_arg_direct(cA + p * CW, rr);
                idx[k] = (pass <= 16) ? p * 32 + r : -1;
            }
#pragma unroll
            for (int k = 0; k < 2; ++k) arg[k] = exp_cap_tab64(arg[k], etab64);
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                if (idx[k] >= 0) {
                    if constexpr (SGN) { if (idx[k] >= 32) arg[k] *= sx; }
                    mB[idx[k]] = arg[k];
                }
            }
        }
        if (tht) ph_s[4] += clock64() - ht0;
        {   // ---- base(K+1)
            const int B = K + 1;
            const double *cA = ctab_s + ((K + 1) & 1) * (4 * 32 * CW), *rA = rtab_s + ((K + 1) & 1) * (2 * 32 * RW) + lane * RW;
            double rt[8];
            ld_entry(rA, rt, (D + 2) / 2);
            // both older column blocks as one batch, so that eight independent exponentials are in flight
            double arg[2][SPEC_NCOL], z[2][SPEC_NCOL];
#pragma unroll
            for (int qq = 0; qq < 2; ++qq) {
                const int q = 2 + qq, C = B - q;
                const bool valid = q <= L && C >= 0;
#pragma unroll
                for (int k = 0; k < SPEC_NCOL; ++k) {
                    const int p = min(hw + SPEC_NHW * k, 31), slot = (C * 32 + p) & (RB - 1);
                    arg[qq][k] = valid ? entry_arg(cA + (q * 32 + p) * CW, rt) : -1e4;
                    z[qq][k] = (valid && hw + SPEC_NHW * k < 32) ? ring_Z[slot] : 0.0;
                }
            }
            const bool live0 = batch_is_live(arg[0]), live1 = batch_is_live(arg[1]);
            if (phase != nullptr && dir == 0 && lane == 0 && K >= 1) { // profiling: batches met / skipped (all helper warps)
                const bool two = L >= 3 && K >= 2;
                atomicAdd(reinterpret_cast<unsigned long long *>(&ph_s[11]), two ? 2ull : 1ull);
                atomicAdd(reinterpret_cast<unsigned long long *>(&ph_s[12]), (live0 ? 0ull : 1ull) + ((two && !live1) ? 1ull : 0ull));
            }
            if (!fact && (live0 || live1)) { // live batches get their arguments the direct way
                double rr[8];
                ld_entry(rA, rr, (2 + 2 * D) / 2);
#pragma unroll
                for (int qq = 0; qq < 2; ++qq) {
                    if (qq ? live1 : live0) {
#pragma unroll
                        for (int k = 0; k < SPEC_NCOL; ++k)
                            arg[qq][k] = entry_arg_direct(cA + ((2 + qq) * 32 + min(hw + SPEC_NHW * k, 31)) * CW, rr);
                    }
                }
            }
            if (live0 && live1) {
#pragma unroll
                for (int k = 0; k < 2 * SPEC_NCOL; ++k) arg[k / SPEC_NCOL][k % SPEC_NCOL] = exp_cap_tab64(arg[k / SPEC_NCOL][k % SPEC_NCOL], etab64);
            } else {
#pragma unroll
                for (int qq = 0; qq < 2; ++qq) {
                    if (qq ? live1 : live0) {
#pragma unroll
                        for (int k = 0; k < SPEC_NCOL; ++k) arg[qq][k] = exp_cap_tab64(arg[qq][k], etab64);
                    } else {
#pragma unroll
                        for (int k = 0; k < SPEC_NCOL; ++k) arg[qq][k] = 0.0;
                    }
                }
            }
#pragma unroll
            for (int qq = 0; qq < 2; ++qq) {
                double sum = 0.0;
#pragma unroll
                for (int k = 0; k < SPEC_NCOL; ++k) sum = fma(z[qq][k], arg[qq][k], sum);
                baseT_s[(((B & 1) * 2 + qq) * SPEC_NHW + hw) * 32 + lane] = sum;
            }
        }
        if (tht) ph_s[5] += clock64() - ht0;
        {   // ---- E'(K+2)
            const int B = K + 2;
            const double *cA = ctab_s + ((K + 1) & 1) * (4 * 32 * CW) + 32 * CW, *rA = rtab_s + ((K + 1) & 1) * (2 * 32 * RW) + (32 + lane) * RW;
            double rt[8];
            ld_entry(rA, rt, (D + 2) / 2);
            double *uB = ue_s + (B & 1) * 1024;
            double arg[SPEC_NCOL];
#pragma unroll
            for (int k = 0; k < SPEC_NCOL; ++k) {
                const int p = min(hw + SPEC_NHW * k, 31);
                arg[k] = entry_arg(cA + p * CW, rt);
            }
            // entries below e^-260 of the row's gauge are nothing (the sums they enter are O(1) in that gauge, give or
            // take the drift of a stale gauge): when a whole batch is that small -- the usual case for blocks of
            // particles that are not neighbours in space -- the exponentials are skipped (warp-uniform)
            const bool live = batch_is_live(arg);
            if (phase != nullptr && dir == 0 && lane == 0 && K >= 0) {
                atomicAdd(reinterpret_cast<unsigned long long *>(&ph_s[11]), 1ull);
                atomicAdd(reinterpret_cast<unsigned long long *>(&ph_s[12]), live ? 0ull : 1ull);
            }
            if (live) {
                if (!fact) {
                    double rr[8];
                    ld_entry(rA, rr, (2 + 2 * D) / 2);
#pragma unroll
                    for (int k = 0; k < SPEC_NCOL; ++k) arg[k] = entry_arg_direct(cA + min(hw + SPEC_NHW * k, 31) * CW, rr);
                }
#pragma unroll
                for (int k = 0; k < SPEC_NCOL; ++k) arg[k] = exp_cap_tab64(arg[k], etab64);
            } else {
#pragma unroll
                for (int k = 0; k < SPEC_NCOL; ++k) arg[k] = 0.0;
            }
#pragma unroll
            for (int k = 0; k < SPEC_NCOL; ++k) {
                const int p = hw + SPEC_NHW * k;
                if (p < 32) {
                    if constexpr (SGN) { if (p >= 1) arg[k] *= sx; }
                    uB[p * 32 + lane] = arg[k];
                }
            }
        }
    };
    // the workers' panel of block B (columns < 32 (B-L), published relative to the T of column 32 (B-L)),
    // scaled like the rest; one warp, lane = row; waits for the workers
    auto fetch_panel = [&](int B) {
        const int b3 = B & 7, jrec0 = 32 * (B - L);
        double v = 0.0;
        if (jrec0 > 0 && B < NBk) {
            const int i = B * 32 + lane;
            if (i < N) {
                const double shift = dd_diff(ring_T[jrec0 & (RB - 1)], trefn_s[b3]) - G_s[b3 * 32 + lane];
                unsigned long long um, us;
                int npoll = 0;
                do { // each lane waits for its own row (k_prep emptied the words, the worker fills them)
                    um = ld_relaxed_u64(&rshift(a.p.pan_m[dir], roff)[i]);
                    us = ld_relaxed_u64(&rshift(a.p.pan_s[dir], roff)[i]);
                    ++npoll;
                } while (um == PAN_EMPTY || us == PAN_EMPTY);
                if (lane == 0 && phase != nullptr && dir == 0) ph_s[10] += npoll; // 1 per block = never waited
                v = __longlong_as_double((long long)us) * exp_cap_tab64(__longlong_as_double((long long)um) + shift, etab64);
            }
        }
        baseP_s[(B & 1) * 32 + lane] = v;
    };
    // 2^e as a double, 0 for e < -1000 (a contribution that far down is nothing), e <= 1000 assumed
    auto pow2i = [](int e) { return e < -1000 ? 0.0 : __hiloint2double((1023 + min(e, 1000)) << 20, 0); };

    // ---- prologue: raw data of blocks 0..3, gauges of blocks 0..2, then the helpers' window "-1"
    for (int B = 0; B < 4; ++B) load_raw(B, tid, CH_THREADS);
    if (tid == 0) {
        const double2 T0 = ldcg2(&g[0]);
        trefn_s[0] = T0;
        ring_T[0] = T0;
        ring_Z[0] = 1.0;
    }
    for (int e = tid; e < 2 * 2 * SPEC_NHW * 32; e += CH_THREADS) baseT_s[e] = 0.0;
    for (int e = tid; e < 2 * 1024; e += CH_THREADS) mt_s[e] = 0.0;
    if (tid < 64) baseP_s[tid] = 0.0;
    if (tid < 8) kacc_s[tid] = 0;
    for (int B = 0; B < 3; ++B) {
        __syncthreads();
        if (warp == 0) gauges(B);
    }
    __syncthreads();
    if (warp == 1) col_row_terms(-2);
    if (warp == 2) col_row_terms(-1);
    __syncthreads();
    if (warp < SPEC_NHW) helper_tasks(-1, warp);

    int bad = 0;                     // warp 0: a row sum of its rows left the acceptance band of the stale gauge
    int kacc = 0;                    // warp 0: power of two taken out of Zhat up to the start of block K
    int kh1 = 0, kh2 = 0, kh3 = 0, kh4 = 0; // warp 0: the same for blocks K-1 .. K-4
    double z0 = 1.0, acc_next = 0.0; // warp 0: Zhat of the block's first column; start value of the next block
    double2 fin_T = make_double2(0.0, 0.0);
    double fin_G = 0.0, fin_acc = 1.0;
    const double2 LN2 = make_double2(0.6931471805599453, 2.3190468138462996e-17);

    const bool tim = phase != nullptr && dir == 0 && tid == 0;
    if (tid < 16) ph_s[tid] = 0;
    long long tprev = clock64();
#define PH(k) do { if (tim) { const long long c__ = clock64(); ph_s[k] += c__ - tprev; tprev = c__; } } while (0)

    for (int K = 0; K < NBk; ++K) {
        __syncthreads(); // everything block K needs is ready; everything of block K-1 has been consumed
        PH(0);
        const int i0 = K * 32, cur = K & 1;
        const int nrows = min(32, N - i0);
        if (warp == 0) {
            const double *mK = mt_s + cur * 1024 + lane, *uN = ue_s + (cur ^ 1) * 1024 + lane;
            // earlier columns, each group brought from its own frame to this block's (exact powers of two);
            // all loads first, the frames of the last blocks are kept in registers (kh[q] = frame of block K-q)
            const double *bq = baseT_s + (cur * 2 * SPEC_NHW) * 32 + lane;
            double b2s = 0.0, b3s = 0.0, b2t = 0.0, b3t = 0.0; // loads are independent, two add chains each
#pragma unroll
            for (int k = 0; k < SPEC_NHW; k += 2) {
                b2s += bq[k * 32];
                b3s += bq[(SPEC_NHW + k) * 32];
                if (k + 1 < SPEC_NHW) { b2t += bq[(k + 1) * 32]; b3t += bq[(SPEC_NHW + k + 1) * 32]; }
            }
            b2s += b2t;
            b3s += b3t;
            const double bp = baseP_s[cur * 32 + lane];
            double m_n = mK[0], u_n = uN[32];
            const double u0 = uN[0];
            double acc = acc_next * pow2i(kh1 - kacc);
            if (K >= 2) acc = fma(b2s, pow2i(kh2 - kacc), acc);
            if (L >= 3 && K >= 3) acc = fma(b3s, pow2i(kh3 - kacc), acc);
            if (K - L - 1 >= 0) acc = fma(bp, pow2i((L == 1 ? kh2 : (L == 2 ? kh3 : kh4)) - kacc), acc);
            double zc = z0;
            acc_next = u0 * z0;
            PH(1);
#pragma unroll
            for (int p = 0; p < 32; ++p) {
                const double m_p = m_n, u_p = u_n; // operands of this step were loaded one step ahead
                if (p < 31) m_n = mK[(p + 1) * 32];
                if (p < 30) u_n = uN[(p + 2) * 32];
                acc = fma(m_p, zc, acc);          // M[p][r] = 0 once p > r
                zc = shfl_bcast(acc, p);          // X^_p; Zhat_{p+1} = sx X^_p (sx is folded into M and E')
                if (p < 31) acc_next = fma(u_p, zc, acc_next);
            }
            PH(2);
            // Zhat of the columns this block produced (frame of block K); the next block's frame takes the
            // exponent of its first column out, so that Zhat stays O(1) however far the solution has drifted
            const double zmine = SGN ? sx * acc : acc;
            const double z32 = SGN ? sx * zc : zc;
            const int ex = (__double2hiint(z32) >> 20) & 0x7ff;
            const int kstep = (ex != 0 && ex != 0x7ff) ? ex - 1023 : 0;
            z0 = z32 * pow2i(-kstep);
            zmail_s[cur * 32 + lane] = zmine;
            const int jn = i0 + lane + 1;
            if (jn < N) ring_Z[jn & (RB - 1)] = (lane == 31) ? z0 : zmine;
            if (lane == 0) kacc_s[K & 7] = kacc;
            // Acceptance band of the stale gauge (DESIGN.md 5.1 "error budget"): every row sum, taken in its block's frame,
            // must lie within 2^+-64 of the gauge (0, NaN and inf fail too; a zero under a stale gauge is a misfit, the
            // max-plus pass decides whether it is a node).  Between two MD steps the solution drifts by e^{+-10} within a
            // block of a spread-out cloud, with a heavy tail from index neighbours that sit far apart (measured: a band
            // of 2^+-8 rejected every step of cfg3, 2^+-32 one step in three at N = 40000); the frames take the drift
            // from block to block.  The helpers drop entries below e^-260 of the row's gauge; with |Zhat| <= 2^64, the
            // frames of the three blocks behind at most 2^192 apart and the row sum itself >= 2^-64 a dropped entry is
            // below e^-260 2^320 = 2e-17 of the row sum.
            if (lane < nrows && !(fabs(acc) > 0x1p-64 && fabs(acc) < 0x1p64)) bad = 1;
            if (K + 1 == NBk) {
                fin_T = dd_add_d(dd_add_d(trefn_s[K & 7], (double)kacc * LN2.x), (double)kacc * LN2.y);
                fin_G = G_s[(K & 7) * 32 + lane];
                fin_acc = acc;
            }
            kh4 = kh3; kh3 = kh2; kh2 = kh1; kh1 = kacc;
            kacc += kstep;
            PH(3);
        } else if (warp == CH_WARPS - 1) {
            const long long hcp = clock64();
            if (K > 0) { // publish the columns block K-1 produced, in its frame (column N is kept too: its T is
                         // the last row's gauge next time)
                const int jn = i0 - 32 + lane + 1;
                if (jn <= N) {
                    const double kf = (double)kacc_s[(K - 1) & 7];
                    g[jn] = dd_add_d(dd_add_d(ring_T[jn & (RB - 1)], kf * LN2.x), kf * LN2.y);
                    gs[jn] = zmail_s[(cur ^ 1) * 32 + lane];
                }
            }
            if (K > 0) {
                __syncwarp();
                if (lane == 0) st_release(&rshift(a.p.cols_ready, roff)[dir], min(N, i0 + 1));
            }
            if (phase != nullptr && dir == 0 && lane == 0) ph_s[7] += clock64() - hcp;
        } else if (warp == CH_WARPS - 3) {
            // gauges of block K+3 (its raw data arrived during the previous window), then the raw data of block K+4
            const long long hcg = clock64();
            gauges(K + 3);
            const int b3 = (K + 4) & 7, i = (K + 4) * 32 + lane;
            double2 told = make_double2(0.0, 0.0), told32 = told;
            Vec<D> pr, pc;
#pragma unroll
            for (int c = 0; c < D; ++c) { pr.v[c] = 0.0; pc.v[c] = 0.0; }
            double c0 = 0.0;
            told = ldcg2(&g[min(i, N)]); // flat beyond the last column (see load_raw)
            if (lane == 0) told32 = ldcg2(&g[min(i + 32, N)]);
            if (i < N) {
                pr = ldvec<D>(rho, i);
                pc = ldvec<D>(sig, i);
                if (i < N - 1) c0 = cc[i];
            }
            __syncwarp(); // G of block K+3 is in place
            col_row_terms(K); // while the loads are in flight
            traw_s[b3 * 34 + lane] = told;
            if (lane == 0) traw_s[b3 * 34 + 32] = told32;
#pragma unroll
            for (int c = 0; c < D; ++c) {
                rho_s[(b3 * 32 + lane) * D + c] = pr.v[c];
                ring_sig[(i & (RB - 1)) * D + c] = pc.v[c];
            }
            cc_s[b3 * 32 + lane] = c0;
            if (phase != nullptr && dir == 0 && lane == 0) ph_s[15] += clock64() - hcg;
        } else if (warp == CH_WARPS - 2) {
            long long hc0 = clock64();
            fetch_panel(K + 1);
            if (phase != nullptr && dir == 0 && lane == 0) ph_s[9] += clock64() - hc0;
        } else if (SPEC_NHW == 12 || (warp & 3) != 0) {
            // helper warps: with SPEC_NHW = 9 the three that share warp 0's scheduler partition (4, 8, 12) stay idle
            const int hw = (SPEC_NHW == 12) ? warp - 1 : warp - 1 - (warp >> 2);
            const bool th = phase != nullptr && dir == 0 && lane == 0 && hw == 0;
            const long long hc0 = clock64();
            helper_tasks(K, hw);
            if (th) ph_s[8] += clock64() - hc0;
            if (phase != nullptr && dir == 0 && lane == 0 && hw == 4) ph_s[13] += clock64() - hc0;
            if (phase != nullptr && dir == 0 && lane == 0 && hw == 8) ph_s[14] += clock64() - hc0;
        }
    }
    __syncthreads();
#undef PH
    if (tim) {
        for (int k = 0; k < 16; ++k) phase[k] += (unsigned long long)ph_s[k];
    }
    if (warp == 0) {
        if (lane == (N - 1) % 32) {
            rshift(a.p.rfin, roff)[dir] = dd_add_d(dd_add_d(fin_T, fin_G), log(fabs(fin_acc)));
            rshift(a.p.rsgn, roff)[dir] = (fin_acc < 0.0) ? -1.0 : 1.0;
        }
        if (bad) atomicOr(a.gauge_misfit, 1);
    }
    if (warp == CH_WARPS - 1) {
        const int jn = (NBk - 1) * 32 + lane + 1;
        if (jn <= N) {
            const double kf = (double)kacc_s[(NBk - 1) & 7];
            g[jn] = dd_add_d(dd_add_d(ring_T[jn & (RB - 1)], kf * LN2.x), kf * LN2.y);
            gs[jn] = zmail_s[((NBk - 1) & 1) * 32 + lane];
        }
        // no fence: bar.warp.sync + st.release.gpu is cumulative over the other lanes' stores
        __syncwarp();
        if (lane == 0) st_release(&rshift(a.p.cols_ready, roff)[dir], N);
    }
}

template <int D, bool SGN>
__device__ void worker_cta(const ChainArgs &a, int dir, int widx, size_t roff, unsigned char *smem_raw, const double *etab64)
{
    const int N = a.N, LOOK = a.look;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // per-warp staging of one column tile: g (dd), sign, sig
    double2 *st_g = reinterpret_cast<double2 *>(smem_raw) + warp * 32;
    double *st_sg = reinterpret_cast<double *>(reinterpret_cast<double2 *>(smem_raw) + CH_WARPS * 32) + warp * 32;
    double *st_sig = reinterpret_cast<double *>(reinterpret_cast<double2 *>(smem_raw) + CH_WARPS * 32) + CH_WARPS * 32 + warp * 32 * D;
    double *mg_m = reinterpret_cast<double *>(reinterpret_cast<double2 *>(smem_raw) + CH_WARPS * 32) + CH_WARPS * 32 + CH_WARPS * 32 * D;
    double *mg_s = mg_m + CH_WARPS * 32;
    double *mg_q = mg_s + CH_WARPS * 32; // [D + 1][CH_WARPS * 32]

    const double *rho = rshift(a.p.rho[dir], roff), *sig = rshift(a.p.sig[dir], roff);
    const double2 *g = rshift(a.p.g[dir], roff);
    const double *gs = rshift(a.p.gs[dir], roff);
    const int *cols_ready = &rshift(a.p.cols_ready, roff)[dir];
    const double kk = a.kk;
    int known_ready = 0;

    for (int K = LOOK + 1 + widx; K < a.NB; K += a.nworkers) {
        const int i = K * 32 + lane;
        Vec<D> pr;
#pragma unroll
        for (int c = 0; c < D; ++c) pr.v[c] = 0.0;
        if (i < N) pr = ldvec<D>(rho, i);
        // exponent arguments in 1 + D instructions per entry, as in chain_cta_spec: with the origin o = row 0 of the
        // block, rho' = rho_r - o, sigma' = sigma_p - o:  (T_p - T_ref) - kk |rho_r - sigma_p|^2 = A_p + B_r +
        // sum_c (2 kk rho'_c) sigma'_c,  A_p = (T_p - T_ref) - kk |sigma'_p|^2 (per column, at staging),
        // B_r = -kk |rho'_r|^2 (per row, here)
        const Vec<D> org = ldvec<D>(rho, K * 32);
        double rowB = 0.0, roww[D], rowp[D];
#pragma unroll
        for (int c = 0; c < D; ++c) {
            const double rp = pr.v[c] - org.v[c];
            rowB = fma(rp, rp, rowB);
            roww[c] = 2.0 * kk * rp;
            rowp[c] = rp;
        }
        rowB *= -kk;
        // the factorised form only while its terms are small (see chain_cta_spec, FACT_LIMIT); decided per chunk
        const bool rows_small = __any_sync(0xffffffffu, i < N && !(-rowB < FACT_LIMIT)) == 0;
        const int ntile = K - LOOK;
        Lse acc = lse_empty();
        // the terms w = Zhat_p exp(tau - m) of the row sum are the very weights of Eq. 15/16 (up to a factor
        // per row that the other direction's table fixes afterwards), so sum w sigma_p and sum w beta C ride along: the
        // panel's share of the exterior forces and of <E_c> costs D + 3 more FP64 instructions per entry here instead of a
        // second sweep with one more exponential per entry (k_forcepass then covers only the LOOK + 1 newest column blocks)
        double tq[D + 1];
#pragma unroll
        for (int c = 0; c < D + 1; ++c) tq[c] = 0.0;
        double2 ref = make_double2(0.0, 0.0);
        // unit of work = 8 columns; chunk c goes to warp c mod 16, so the four chunks of the newest tile (the
        // ones the chain is waiting for) are done by four warps at once
        // The columns of the next chunk are loaded (registers of lanes 0..7) while the current one is computed:
        // an L2 round trip is ~800 cycles, a chunk ~300.
        double2 pre_g = make_double2(0.0, 0.0);
        double pre_z = 0.0;
        Vec<D> pre_c;
#pragma unroll
        for (int c = 0; c < D; ++c) pre_c.v[c] = 0.0;
        bool have_pre = false, col_big = false;
        auto cols_are_ready = [&](int c8, bool wait) {
            const int need = 32 * ((c8 >> 2) + 1);
            if (known_ready < need) {
                if (lane == 0) {
                    int v = ld_acquire(cols_ready);
                    while (wait && v < need) v = ld_acquire(cols_ready);
                    known_ready = v;
                }
                known_ready = __shfl_sync(0xffffffffu, known_ready, 0);
            }
            return known_ready >= need;
        };
        // lane 8 of a warp that takes a chunk of the newest tile also fetches column 32 ntile, the reference the
        // panel is published against (cols_ready is 32 K' + 1 or N, so that column came with the same publication)
        double2 pub_pre = make_double2(0.0, 0.0);
        bool have_pub = false;
        auto load_cols = [&](int c8) {
            if (lane < 8) {
                const int j = 8 * c8 + lane;
                pre_g = ldcg2(&g[j]);
                pre_z = ldcg1(&gs[j]);
                pre_c = ldvec<D>(sig, j);
            }
            if ((c8 >> 2) == ntile - 1) {
                if (lane == 8) pub_pre = ldcg2(&g[32 * ntile]);
                have_pub = true;
            }
        };
        for (int c8 = warp; c8 < 4 * ntile; c8 += CH_WARPS) {
            if (!have_pre) {
                cols_are_ready(c8, true);
                load_cols(c8);
            }
            __syncwarp();
            {
                // the chunk's first column is its reference; every column leaves (A_p, sigma'_p, Zhat_p)
                const double2 g0 = make_double2(shfl_bcast(pre_g.x, 0), shfl_bcast(pre_g.y, 0));
                col_big = false;
                if (lane < 8) {
                    double n2 = 0.0;
#pragma unroll
                    for (int c = 0; c < D; ++c) {
                        const double sp = pre_c.v[c] - org.v[c];
                        n2 = fma(sp, sp, n2);
                        st_sig[lane * D + c] = sp;
                    }
                    const double td = dd_diff(pre_g, g0);
                    st_g[8 + lane] = make_double2(fma(-kk, n2, td), td);
                    st_sg[lane] = pre_z;
                    if (lane == 0) st_g[0] = pre_g;
                    col_big = !(kk * n2 + fabs(td) < FACT_LIMIT);
                }
            }
            const bool fact = rows_small && __any_sync(0xffffffffu, col_big) == 0;
            __syncwarp();
            have_pre = (c8 + CH_WARPS < 4 * ntile) && cols_are_ready(c8 + CH_WARPS, false);
            if (have_pre) load_cols(c8 + CH_WARPS);
            const double2 nref = st_g[0];
            lse_shift(acc, dd_diff(ref, nref));
            ref = nref;
            double tau[8];
            if (fact) {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    double t = st_g[8 + k].x + rowB;
#pragma unroll
                    for (int c = 0; c < D; ++c) t = fma(roww[c], st_sig[k * D + c], t);
                    tau[k] = t;
                }
            } else {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    double dd = rowp[0] - st_sig[k * D];
                    double r2 = dd * dd;
#pragma unroll
                    for (int c = 1; c < D; ++c) { dd = rowp[c] - st_sig[k * D + c]; r2 = fma(dd, dd, r2); }
                    tau[k] = fma(-kk, r2, st_g[8 + k].y);
                }
            }
            // maximum as a tree (three levels instead of a chain of eight)
            const double cm = fmax(fmax(fmax(tau[0], tau[1]), fmax(tau[2], tau[3])), fmax(fmax(tau[4], tau[5]), fmax(tau[6], tau[7])));
            if (cm > acc.m) {
                const double f = exp_neg_tab64(-(acc.m - cm), etab64);
                acc.s *= f;
#pragma unroll
                for (int c = 0; c < D + 1; ++c) tq[c] *= f;
                acc.m = cm;
            }
            double s0 = 0.0, s1 = 0.0, q0[D + 1], q1[D + 1];
#pragma unroll
            for (int c = 0; c < D + 1; ++c) { q0[c] = 0.0; q1[c] = 0.0; }
#pragma unroll
            for (int k = 0; k < 8; k += 2) {
                const double w0 = exp_neg_tab64(-(tau[k] - acc.m), etab64) * st_sg[k];
                const double w1 = exp_neg_tab64(-(tau[k + 1] - acc.m), etab64) * st_sg[k + 1];
                s0 += w0;
                s1 += w1;
#pragma unroll
                for (int c = 0; c < D; ++c) {
                    q0[c] = fma(w0, st_sig[k * D + c], q0[c]);
                    q1[c] = fma(w1, st_sig[(k + 1) * D + c], q1[c]);
                }
                // beta C = kk |rho - sigma|^2 = (T_p - T_ref) - tau
                q0[D] = fma(w0, st_g[8 + k].y - tau[k], q0[D]);
                q1[D] = fma(w1, st_g[8 + k + 1].y - tau[k + 1], q1[D]);
            }
            acc.s += s0 + s1;
#pragma unroll
            for (int c = 0; c < D + 1; ++c) tq[c] += q0[c] + q1[c];
            __syncwarp();
        }
        // common reference of the published partial: g_{32 ntile} (first "recent" column of block K)
        if (have_pub) {
            const double2 pub = make_double2(shfl_bcast(pub_pre.x, 8), shfl_bcast(pub_pre.y, 8));
            lse_shift(acc, dd_diff(ref, pub));
        } else {
            const int need = 32 * ntile + 1;
            if (known_ready < need) {
                if (lane == 0) {
                    int v;
                    while ((v = ld_acquire(cols_ready)) < need) { }
                    known_ready = v;
                }
                known_ready = __shfl_sync(0xffffffffu, known_ready, 0);
            }
            __syncwarp();
            const double2 pub = ldcg2(&g[32 * ntile]);
            lse_shift(acc, dd_diff(ref, pub));
        }
        mg_m[warp * 32 + lane] = acc.m;
        mg_s[warp * 32 + lane] = acc.s;
#pragma unroll
        for (int c = 0; c < D + 1; ++c) mg_q[(c * CH_WARPS + warp) * 32 + lane] = tq[c];
        __syncthreads();
        if (warp == 0) {
            // 16 partials per row: maximum first, then 16 independent exponentials
            Lse t = lse_empty();
#pragma unroll
            for (int w = 0; w < CH_WARPS; ++w) t.m = fmax(t.m, mg_m[w * 32 + lane]);
            double fw[CH_WARPS];
#pragma unroll
            for (int w = 0; w < CH_WARPS; ++w) fw[w] = 0.0;
            if (t.m > -INFINITY) {
#pragma unroll
                for (int w = 0; w < CH_WARPS; ++w) {
                    fw[w] = exp_neg_tab64(-(mg_m[w * 32 + lane] - t.m), etab64);
                    t.s = fma(mg_s[w * 32 + lane], fw[w], t.s);
                }
            }
            if (i < N) { // the chain is waiting for these two words
                st_relaxed_f64(&rshift(a.p.pan_m[dir], roff)[i], t.m);
                st_relaxed_f64(&rshift(a.p.pan_s[dir], roff)[i], t.s);
            }
            // no fence: bar.warp.sync + st.release.gpu is cumulative over the other lanes' stores
            __syncwarp();
            if (lane == 0) st_release(&rshift(a.p.panel_ready[dir], roff)[K], 1);
            // the force sums of the panel, same units (k_assemble scales them); sigma' was taken about the block's origin
            if (i < N) {
                double *pq = rshift(a.p.pacc[dir], roff) + (size_t)i * (D + 1);
#pragma unroll
                for (int c = 0; c < D + 1; ++c) {
                    double q = 0.0;
#pragma unroll
                    for (int w = 0; w < CH_WARPS; ++w) q = fma(mg_q[(c * CH_WARPS + w) * 32 + lane], fw[w], q);
                    pq[c] = (c < D) ? fma(org.v[c < D ? c : 0], t.s, q) : q;
                }
            }
        }
        __syncthreads();
    }
}

template <int D> size_t chain_spec_smem_bytes_host()
{
    const size_t chain = SpecSmem<D>().total * 8;
    const size_t worker = (size_t)CH_WARPS * 32 * (16 + 8 + D * 8) + (size_t)CH_WARPS * 32 * 16 + (size_t)CH_WARPS * 32 * 8 * (D + 1);
    return chain > worker ? chain : worker;
}

// ==========================================================================================
// Step 6: connection probabilities (Eq. 12) and the sums the
// exterior-bead forces need (Eq. 15, 16), no N x N storage:
//   Pr[l -> l'] = sg exp( qhat[l] + a[l'] - kk |r_l^P - r_l'^1|^2 - R_N ),  l' <= l
// In generic form, for direction dir and row i:
//   w_ij = exp( g^{other}[N-1-i] + g^{dir}[j] - kk |rho_i - sig_j|^2 - R_N ),  j <= i
//   acc[dir][i] = ( sum_j w, sum_j w sig_j, sum_j w kk r2 )
// dir 0 gives the row sums (bead P, Eq. 16), dir 1 the column sums (bead 1, Eq. 15).
// The terms w_ij are, up to a factor per row, the terms of the recursion's own row sums: the panel
// workers accumulate sum w sig and sum w kk r2 over all columns older than the LOOK newest blocks while they form the
// panel (p.pacc), so forceband_task covers only the near-diagonal band of (LOOK + 1) column blocks per row block:
// N (LOOK + 1) 32 entries per direction instead of N^2/2.  One task per row block and direction, run by groups of 128
// threads in the tail of the recursion kernels (exchange_tail).
// ==========================================================================================

template <int D, bool SGN>
__device__ void forceband_task(int N, double kk, const ExchPtrs &p, int band, int rt, int dir, int tid, int bar_id, double *sm,
                               const double *etab)
{
    // A group of FP_TB = 128 threads (tid = 0..127, its own named barrier) takes one block of RT = 32 rows and the
    // (band + 1) <= 4 newest column blocks of it, the ones the recursion kept inside its chain CTA (columns
    // j0 = 32 (K - band) .. i); the sums over all older columns come from the panel workers (p.pacc, added in
    // assemble_task).  Four threads per row with 32 columns each, partial sums combined in shared memory.  Every row is
    // written by exactly one group: plain stores.
    constexpr int NQ = 4, CW = FP_TB / NQ, RT = FP_TB / NQ;
    const int j0 = max(0, 32 * (rt - band));
    double2 *sg_g = reinterpret_cast<double2 *>(sm);
    double *sg_s = sm + 2 * FP_TB, *sg_sig = sg_s + FP_TB, *part_s = sg_sig + FP_TB * D;
    const double2 *gd = p.g[dir], *go = p.g[1 - dir];
    const int r = tid % RT, q = tid / RT;
    const int i = rt * RT + r;
    bar_sync_named(bar_id, FP_TB); // the previous task of this group is done with the staging area
    {
        const int j = j0 + tid;
        double2 gj = make_double2(-INFINITY, 0.0);
        double sj = 1.0;
        Vec<D> sc;
#pragma unroll
        for (int c = 0; c < D; ++c) sc.v[c] = 0.0;
        if (j < N) {
            gj = gd[j];
            sj = p.gs[dir][j];
            sc = ldvec<D>(p.sig[dir], j);
        }
        sg_g[tid] = gj;
        sg_s[tid] = sj;
#pragma unroll
        for (int c = 0; c < D; ++c) sg_sig[tid * D + c] = sc.v[c];
    }
    bar_sync_named(bar_id, FP_TB);
    const int k0 = q * CW;
    const int ncol = (i < N) ? min(CW, i - (j0 + k0) + 1) : 0; // columns j0+k0 .. min(j0+k0+CW-1, i)
    double sw = 0.0, swc = 0.0, osg = 0.0;
    Vec<D> sws;
#pragma unroll
    for (int c = 0; c < D; ++c) sws.v[c] = 0.0;
    if (ncol > 0) {
        const Vec<D> pr = ldvec<D>(p.rho[dir], i);
        // A = g^{other}[N-1-i] - R_N as dd, rounded once per element after adding g^{dir}[j]
        const double2 A = dd_sub(go[N - 1 - i], p.rfin[0]);
        osg = p.gs[1 - dir][N - 1 - i];
        if constexpr (SGN) osg *= p.rsgn[0];
#pragma unroll 4
        for (int k = k0; k < k0 + ncol; ++k) {
            Vec<D> pc;
#pragma unroll
            for (int c = 0; c < D; ++c) pc.v[c] = sg_sig[k * D + c];
            const double2 gj = sg_g[k];
            const double kr2 = kk * dist2<D>(pr, pc);
            const double targ = ((A.x + gj.x) + (A.y + gj.y)) - kr2;
            const double w = exp_cap_tab64(targ, etab) * sg_s[k];
            sw += w;
            swc = fma(w, kr2, swc);
#pragma unroll
            for (int c = 0; c < D; ++c) sws.v[c] = fma(w, pc.v[c], sws.v[c]);
        }
    }
    part_s[(q * (D + 2)) * RT + r] = osg * sw;
#pragma unroll
    for (int c = 0; c < D; ++c) part_s[(q * (D + 2) + 1 + c) * RT + r] = osg * sws.v[c];
    part_s[(q * (D + 2) + D + 1) * RT + r] = osg * swc;
    bar_sync_named(bar_id, FP_TB);
    // thread (r, q) adds up components q, q + NQ, .. of row r
    if (i < N) {
        for (int c = q; c < D + 2; c += NQ) {
            double t = 0.0;
#pragma unroll
            for (int qq = 0; qq < NQ; ++qq) t += part_s[(qq * (D + 2) + c) * RT + r];
            p.acc[dir][(size_t)i * (D + 2) + c] = t;
        }
    }
}

// ==========================================================================================
// Eq. 13 and the assembly of the exterior forces (Eq. 15, 16):
//   Pr[l -> l+1] = 1 - xi (l+1) sg exp( qhat[l] + a[l+1] - beta C(l,l+1) - R_N )
//   FexP[l] = -k_s ( r_l^P - sum_{l'} Pr[l -> l'] r_l'^1 ),  Fex1[l] = -k_s ( r_l^1 - sum_{l'} Pr[l' -> l] r_l'^P )
// (the intra-ring halves -k_s (r^P - r^{P-1}), -k_s (r^1 - r^2) are in k_bead; rows sum to 1).
// One thread per particle.  ecpart: per-block partial sums of sum_{l'} Pr[l->l'] beta C(l,l').
// ==========================================================================================
template <int D, bool SGN>
__device__ void assemble_task(int N, double ks, double xi, const ExchPtrs &p, double *Fex1, double *FexP, double *ecpart, int band,
                              int chunk, int tid, int bar_id, double *red /* 4 doubles of the group */)
{
    // a group of FP_TB = 128 threads takes the particles [128 chunk, 128 chunk + 128); ecpart[chunk] = their share of <E_c>
    const int l = chunk * FP_TB + tid;
    double ec = 0.0;
    if (l < N) {
        const double2 R = p.rfin[0];
        const double rs_ = SGN ? p.rsgn[0] : 1.0;
        auto pn = [&](int m) -> double { // Pr[m -> m+1], 0 <= m <= N-2
            const double2 A = dd_sub(p.g[1][N - 1 - m], R);
            const double2 B = p.g[0][m + 1];
            const double w = exp_fast(((A.x + B.x) + (A.y + B.y)) - p.cnext[m]) * (p.gs[1][N - 1 - m] * p.gs[0][m + 1] * rs_);
            return 1.0 - xi * (double)(m + 1) * w;
        };
        const double pl = (l < N - 1) ? pn(l) : 0.0;
        const double pm1 = (l > 0) ? pn(l - 1) : 0.0;
        p.pnext[l] = pl;
        const Vec<D> xP = ldvec<D>(p.rho[0], l), x1 = ldvec<D>(p.sig[0], l);
        const double *a0 = p.acc[0] + (size_t)l * (D + 2);
        const double *a1 = p.acc[1] + (size_t)(N - 1 - l) * (D + 2);
        // The panel's share (band >= 0): the workers left, per row i of direction dir, sum_j w_ij (sig_j, beta C_ij) over
        // the columns j < jp = 32 (i/32 - band) with w_ij = Zhat_j exp(T_j - T_jp - kk r^2 - m_i); the weight of Eq. 12 is
        // w_ij Zhat^{other} exp(T_jp + m_i + g^{other}[N-1-i] - R_N)  (the factor a second sweep used to apply entry by entry)
        double pan[2][D + 1];
#pragma unroll
        for (int dir = 0; dir < 2; ++dir) {
            const int i = dir ? N - 1 - l : l, jp = 32 * (i / 32 - band);
#pragma unroll
            for (int c = 0; c < D + 1; ++c) pan[dir][c] = 0.0;
            if (band >= 0 && jp > 0) {
                const double2 A = dd_sub(p.g[1 - dir][N - 1 - i], R), Tp = p.g[dir][jp];
                double f = exp_fast((((A.x + Tp.x) + (A.y + Tp.y)) + p.pan_m[dir][i])) * p.gs[1 - dir][N - 1 - i] * rs_;
                if (!(fabs(f) < INFINITY)) f = 0.0; // an empty panel (m = -inf) has nothing to add
#pragma unroll
                for (int c = 0; c < D + 1; ++c) pan[dir][c] = f * p.pacc[dir][(size_t)i * (D + 1) + c];
            }
        }
        Vec<D> fP, f1;
#pragma unroll
        for (int c = 0; c < D; ++c) {
            double sP = a0[1 + c] + pan[0][c];
            if (l < N - 1) sP = fma(pl, p.sig[0][(size_t)(l + 1) * D + c], sP);
            double s1 = a1[1 + c] + pan[1][c];
            if (l > 0) s1 = fma(pm1, p.rho[0][(size_t)(l - 1) * D + c], s1);
            fP.v[c] = -ks * (xP.v[c] - sP);
            f1.v[c] = -ks * (x1.v[c] - s1);
        }
        stvec<D>(FexP, l, fP);
        stvec<D>(Fex1, l, f1);
        ec = a0[D + 1] + pan[0][D] + pl * p.cnext[l];
    }
    ec = warp_sum(ec);
    bar_sync_named(bar_id, FP_TB);
    if ((tid & 31) == 0) red[tid >> 5] = ec;
    bar_sync_named(bar_id, FP_TB);
    if (tid == 0) ecpart[chunk] = (red[0] + red[1]) + (red[2] + red[3]);
}

// ==========================================================================================
// Tail of the recursion kernels: once both directions are done (grid barrier), the CTAs of a replica share out the
// force-band tasks (one per row block and direction), meet at a second grid barrier and assemble the exterior forces.
// Two launches less on the critical path of a step (k_forcepass, k_assemble used to be kernels of their own:
// profiles/r2_measurements.md).  Groups of 128 threads with their own named barriers (ids 1..4) and staging areas.
// ==========================================================================================
template <int D, bool SGN>
__device__ void exchange_tail(const ChainArgs &a, size_t roff, unsigned char *smem_raw, const double *etab64,
                              cooperative_groups::grid_group &grid)
{
    const int grp = threadIdx.x >> 7, tid = threadIdx.x & 127, bar_id = 1 + grp;
    const int ngrp = CH_THREADS / FP_TB;
    const int cid = blockIdx.x + gridDim.x * blockIdx.y, ncta = gridDim.x * gridDim.y; // the CTAs of this replica
    const ExchPtrs p = rshift(a.p, roff);
    double *sm = reinterpret_cast<double *>(smem_raw) + grp * fp_task_doubles<D>();
    for (int task = cid * ngrp + grp; task < 2 * a.NB; task += ncta * ngrp)
        forceband_task<D, SGN>(a.N, a.kk, p, a.look_fb, task >> 1, task & 1, tid, bar_id, sm, etab64);
    __threadfence();
    grid.sync();
    const double xi = rshift(a.rp, roff)->xi;
    const int nchunk = (a.N + FP_TB - 1) / FP_TB;
    for (int chunk = cid * ngrp + grp; chunk < nchunk; chunk += ncta * ngrp)
        assemble_task<D, SGN>(a.N, a.ks, xi, p, rshift(a.Fex1, roff), rshift(a.FexP, roff), rshift(a.ecpart, roff), a.look_fb, chunk, tid,
                              bar_id, sm);
}


template <int D, bool SGN>
__global__ void __launch_bounds__(CH_THREADS, 1) k_chain(ChainArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double etab[32], etab64[64]; // 2^(i/32), 2^(i/64)
    if (threadIdx.x < 32) etab[threadIdx.x] = c_exp2_32[threadIdx.x];
    if (threadIdx.x < 64) etab64[threadIdx.x] = c_exp2_64[threadIdx.x];
    __syncthreads();
    const int dir = blockIdx.y;
    const size_t roff = (size_t)blockIdx.z * a.rs; // replica of a batch
    if (blockIdx.x == 0) chain_cta<D, SGN>(a, dir, roff, smem_raw, etab);
    else worker_cta<D, SGN>(a, dir, blockIdx.x - 1, roff, smem_raw, etab64);
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    __threadfence();
    grid.sync();
    exchange_tail<D, SGN>(a, roff, smem_raw, etab64, grid);
}

// the recursion with the previous evaluation's gauge (see chain_cta_spec); same grid, same workers
template <int D, bool SGN>
__global__ void __launch_bounds__(CH_THREADS, 1) k_chain_spec(ChainArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double etab[32], etab64[64];
    if (threadIdx.x < 32) etab[threadIdx.x] = c_exp2_32[threadIdx.x];
    if (threadIdx.x < 64) etab64[threadIdx.x] = c_exp2_64[threadIdx.x];
    __syncthreads();
    const int dir = blockIdx.y;
    const size_t roff = (size_t)blockIdx.z * a.rs;
    if (blockIdx.x == 0) chain_cta_spec<D, SGN>(a, dir, roff, smem_raw, etab64);
    else worker_cta<D, SGN>(a, dir, blockIdx.x - 1, roff, smem_raw, etab64);
    // Safety net in the same launch (a second, conditional cooperative launch cost 7 us per evaluation): if a row sum
    // left the band the stale gauge covers (in any replica of the batch), every CTA sees the misfit flag after the grid
    // barrier and the whole grid redoes the recursion with a fresh max-plus gauge (chain_cta), which overwrites everything
    // this pass published.
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    __threadfence();
    grid.sync();
    if (ld_acquire(a.gauge_misfit) != 0) { // the same answer in every CTA
        if (blockIdx.x == 0 && blockIdx.y == 0) {
            int *pr0 = rshift(a.p.panel_ready[0], roff), *pr1 = rshift(a.p.panel_ready[1], roff);
            for (int k = threadIdx.x; k < a.NB; k += CH_THREADS) { pr0[k] = 0; pr1[k] = 0; }
            if (threadIdx.x < 2) rshift(a.p.cols_ready, roff)[threadIdx.x] = 1;
            if (threadIdx.x == 0 && blockIdx.z == 0) atomicAdd(a.fallbacks, 1ull);
        }
        __threadfence();
        grid.sync();
        ChainArgs b = a;
        b.look = a.look_fb;
        b.phase = nullptr;
        if (blockIdx.x == 0) chain_cta<D, SGN>(b, dir, roff, smem_raw, etab);
        else worker_cta<D, SGN>(b, dir, blockIdx.x - 1, roff, smem_raw, etab64);
        __threadfence();
        grid.sync();
    }
    exchange_tail<D, SGN>(a, roff, smem_raw, etab64, grid);
}

// ==========================================================================================
// The paper's N x N intermediates, materialised on request (they are never needed by the hot path,
// which recomputes their entries on the fly):
//   k_emat   E^{[u,v]} = T[v] - S[u-1] + C[v][u], u <= v (Eq. 7-10)
//   k_prmat  Pr[G(l) = l'] (Eq. 12-14) from the tables of a completed evaluation
// Both are pure streaming writes of 8 N^2 bytes (inputs are O(N) and L2 resident): HBM-write bound.
// One CTA per (row, 1024-column segment); consecutive threads write consecutive columns.
// ==========================================================================================
// S[v] = sum_{l<=v} (E_int[l] + C(l,l+1)), T[v] = S[v-1] + E_int[v] (0-based v); one block, any N
__global__ void __launch_bounds__(1024) k_prefix_st(int N, double beta, const double *__restrict__ eint,
                                                    const double *__restrict__ cnext_beta, double *__restrict__ S, double *__restrict__ T)
{
    __shared__ double wsum[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int per = (N + 1023) / 1024, lo = tid * per, hi = min(N, lo + per);
    double loc = 0.0;
    for (int l = lo; l < hi; ++l) loc += eint[l] + cnext_beta[l] / beta;
    double inc = loc; // inclusive scan of the per-thread sums
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double t = shfl_bcast(inc, max(lane - o, 0));
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        double w = wsum[lane], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double t = shfl_bcast(wi, max(lane - o, 0));
            if (lane >= o) wi += t;
        }
        wsum[lane] = wi - w; // exclusive
    }
    __syncthreads();
    double run = wsum[warp] + (inc - loc); // sum of everything before this thread's segment
    for (int l = lo; l < hi; ++l) {
        T[l] = run + eint[l];
        run += eint[l] + cnext_beta[l] / beta;
        S[l] = run;
    }
}

template <int D>
__global__ void __launch_bounds__(256) k_emat(int N, double ks, const double *__restrict__ xP /* rho[0] */,
                                              const double *__restrict__ x1 /* sig[0] */, const double *__restrict__ S,
                                              const double *__restrict__ T, double *__restrict__ E)
{
    const int u = blockIdx.y;
    const int v0 = blockIdx.x * 1024 + threadIdx.x;
    const Vec<D> r1 = ldvec<D>(x1, u);
    const double Sm = (u > 0) ? S[u - 1] : 0.0;
    double *row = E + (size_t)u * N;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int v = v0 + 256 * k;
        if (v < N) {
            double e = 0.0;
            if (v >= u) e = (T[v] - Sm) + 0.5 * ks * dist2<D>(ldvec<D>(xP, v), r1);
            __stcs(row + v, e);
        }
    }
}

constexpr int PRMAT_ROWS = 8; // rows per CTA: the column tables are read once and kept in registers for all of them
constexpr int PRMAT_COLS = 4; // columns per thread (256 apart)
// four CTAs per SM (64 registers) instead of the three that 72 registers allow: N=10000 0.185 -> 0.170 ms; two columns per
// thread (56 registers) measured 0.175, one 0.233, and taking row blocks alternately from the top (zeros) and the bottom
// (exponentials) of the matrix changed nothing: the lower triangle is FP64 bound at the pair kernel's rate
constexpr int PRMAT_MINB = 4;

template <int D, bool SGN>
__global__ void __launch_bounds__(256, PRMAT_MINB) k_prmat(int N, double kk, ExchPtrs p, double *__restrict__ Pr)
{
    __shared__ double etab256[256];
    etab256[threadIdx.x] = g_exp2_256[threadIdx.x];
    __syncthreads();
    const int l0 = blockIdx.y * PRMAT_ROWS;
    const int c0 = blockIdx.x * (256 * PRMAT_COLS) + threadIdx.x;
    if (c0 - threadIdx.x > l0 + PRMAT_ROWS) {
        // the whole segment lies two or more above the diagonal of all these rows: zeros
        for (int r = 0; r < PRMAT_ROWS && l0 + r < N; ++r) {
#pragma unroll
            for (int k = 0; k < PRMAT_COLS; ++k) {
                const int lp = c0 + 256 * k;
                if (lp < N) __stcs(Pr + (size_t)(l0 + r) * N + lp, 0.0);
            }
        }
        return;
    }
    double2 gj[PRMAT_COLS];
    double zj[PRMAT_COLS];
    Vec<D> sj[PRMAT_COLS];
#pragma unroll
    for (int k = 0; k < PRMAT_COLS; ++k) {
        const int lp = min(c0 + 256 * k, N - 1);
        gj[k] = p.g[0][lp];
        zj[k] = p.gs[0][lp];
        sj[k] = ldvec<D>(p.sig[0], lp);
    }
    for (int r = 0; r < PRMAT_ROWS; ++r) {
        const int l = l0 + r;
        if (l >= N) break;
        const Vec<D> rP = ldvec<D>(p.rho[0], l);
        const double2 A = dd_sub(p.g[1][N - 1 - l], p.rfin[0]);
        double osg = p.gs[1][N - 1 - l];
        if constexpr (SGN) osg *= p.rsgn[0];
        const double pn = p.pnext[l];
        double *row = Pr + (size_t)l * N;
        double w[PRMAT_COLS];
#pragma unroll
        for (int k = 0; k < PRMAT_COLS; ++k)
            w[k] = exp_cap_tab256(((A.x + gj[k].x) + (A.y + gj[k].y)) - kk * dist2<D>(rP, sj[k]), etab256);
#pragma unroll
        for (int k = 0; k < PRMAT_COLS; ++k) {
            const int lp = c0 + 256 * k;
            if (lp < N) __stcs(row + lp, lp <= l ? osg * zj[k] * w[k] : (lp == l + 1 ? pn : 0.0));
        }
    }
}

// xi = 0 (0^0 = 1): only k = 1 survives in Eq. 6, Pr is the identity, every ring closes
// on itself.  V = sum_l E^{[l,l]} + (1/beta) ln N!.
template <int D, int TB>
__global__ void __launch_bounds__(TB) k_exch_xi0(int N, double ks, ExchPtrs p, double *Fex1, double *FexP, double *ecpart, size_t rs)
{
    __shared__ double red[TB / 32];
    const size_t off = (size_t)blockIdx.y * rs;
    p = rshift(p, off); Fex1 = rshift(Fex1, off); FexP = rshift(FexP, off); ecpart = rshift(ecpart, off);
    const int l = blockIdx.x * TB + threadIdx.x;
    double ec = 0.0;
    if (l < N) {
        const Vec<D> xP = ldvec<D>(p.rho[0], l), x1 = ldvec<D>(p.sig[0], l);
        Vec<D> fP, f1;
#pragma unroll
        for (int c = 0; c < D; ++c) {
            fP.v[c] = -ks * (xP.v[c] - x1.v[c]);
            f1.v[c] = -ks * (x1.v[c] - xP.v[c]);
        }
        stvec<D>(FexP, l, fP);
        stvec<D>(Fex1, l, f1);
        p.pnext[l] = 0.0;
        ec = p.cself[l];
    }
    double s = block_sum<TB>(ec, red);
    if (threadIdx.x == 0) ecpart[blockIdx.x] = s;
}

// ==========================================================================================
// Scalars of one evaluation: V_xi^{[1,N]} = T_N - (R_N + N lambda - ln N)/beta (from Eq. 6 with the
// de-trended variable), its sign, <E_c> for the primitive estimator.  One block.
// ==========================================================================================
struct Scalars {
    double vb, sign, ec, sum_eint, sum_cnext_beta, pad[3];
};

template <int TB>
__global__ void __launch_bounds__(TB) k_finalize(int N, int nprep, int nasm, double beta, const RepParams *rp,
                                                double lgammaN1, ExchPtrs p, const double *ecpart, Scalars *out, size_t rs)
{
    __shared__ double red[TB / 32];
    const size_t off = (size_t)blockIdx.x * rs; // one block per replica
    p = rshift(p, off); ecpart = rshift(ecpart, off); out = rshift(out, off);
    const double lambda = rshift(rp, off)->lambda, xi = rshift(rp, off)->xi;
    double a = 0.0, b = 0.0, c = 0.0;
    for (int i = threadIdx.x; i < nprep; i += TB) { a += p.tpart[2 * i]; b += p.tpart[2 * i + 1]; }
    for (int i = threadIdx.x; i < nasm; i += TB) c += ecpart[i];
    a = block_sum<TB>(a, red);
    b = block_sum<TB>(b, red);
    c = block_sum<TB>(c, red);
    if (threadIdx.x == 0) {
        out->sum_eint = a;
        out->sum_cnext_beta = b;
        out->ec = a + c / beta;
        if (xi == 0.0) {
            out->vb = a + c / beta + lgammaN1 / beta; // sum_l (E_int + C(l,l)) + ln N!/beta
            out->sign = 1.0;
        } else {
            const double2 R = p.rfin[0];
            const double TN = a + b / beta;
            // L_N = R_N - beta T_N + N lambda - ln N
            out->vb = TN - ((R.x + ((double)N * lambda - log((double)N))) + R.y) / beta;
            const double sx = xi < 0.0 ? -1.0 : 1.0;
            out->sign = p.rsgn[0] * (((N + 1) & 1) ? sx : 1.0);
        }
    }
}

// ==========================================================================================
// Step 7: velocity Verlet + thermostat (R10), fused:
//   [close step s: v += dt/2 F ; thermostat half]  [open step s+1: thermostat half ; v += dt/2 F ; x += dt v]
// One thread per degree of freedom.  F_total = F + exterior exchange forces on beads 1 and P.
// ==========================================================================================
PIMD_DEV void nhc_half(double &vi, double *vx, double h, double kT, double Q)
{
    constexpr int M = 4;
    double G;
    G = (Q * vx[M - 2] * vx[M - 2] - kT) / Q;
    vx[M - 1] += 0.5 * h * G;
#pragma unroll
    for (int k = M - 2; k >= 0; --k) {
        const double a = exp(-0.25 * h * vx[k + 1]);
        G = (k == 0) ? (vi * vi - kT) / Q : (Q * vx[k - 1] * vx[k - 1] - kT) / Q;
        vx[k] = (vx[k] * a + 0.5 * h * G) * a;
    }
    vi *= exp(-h * vx[0]);
#pragma unroll
    for (int k = 0; k <= M - 2; ++k) {
        const double a = exp(-0.25 * h * vx[k + 1]);
        G = (k == 0) ? (vi * vi - kT) / Q : (Q * vx[k - 1] * vx[k - 1] - kT) / Q;
        vx[k] = (vx[k] * a + 0.5 * h * G) * a;
    }
    G = (Q * vx[M - 2] * vx[M - 2] - kT) / Q;
    vx[M - 1] += 0.5 * h * G;
}

// Bead shards: P = local slices; own_first / own_last say whether local slice 0 / P-1 is the ring's bead 1 /
// bead P (only those take the exterior exchange forces); dof0 = global index of local degree of freedom 0, so that the
// noise of a degree of freedom does not depend on how the beads are sharded.  grid (ceil(ndof/256), B).
template <int THERMO>
__global__ void __launch_bounds__(256) k_integrate(double *__restrict__ x, double *__restrict__ v, const double *__restrict__ F,
                                                  const double *__restrict__ Fex1, const double *__restrict__ FexP,
                                                  double *__restrict__ nhc, size_t ndof, size_t slice /* N*d */, int P,
                                                  double dt, double c1, double c2, double beta, double Q, const RepParams *rp,
                                                  uint64_t step_close, uint64_t step_open, int do_close, int do_open,
                                                  int *istatus, const unsigned long long *dstep, int own_first, int own_last,
                                                  size_t dof0, size_t rs)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= ndof) return;
    const size_t off = (size_t)blockIdx.y * rs;
    x = rshift(x, off); v = rshift(v, off); F = rshift(F, off); Fex1 = rshift(Fex1, off); FexP = rshift(FexP, off);
    [[maybe_unused]] const uint64_t seed = rshift(rp, off)->seed;
    // step counter kept on the device when launches are replayed from a CUDA graph (no per-step arguments there)
    [[maybe_unused]] const uint64_t s_close = dstep ? *dstep : step_close;
    [[maybe_unused]] const uint64_t s_open = dstep ? *dstep + (do_close ? 1 : 0) : step_open;
    const size_t j = idx / slice, rem = idx - j * slice;
    double f = F[idx];
    if (j == 0 && own_first) f += Fex1[rem];
    if (j == (size_t)(P - 1) && own_last) f += FexP[rem];
    double vi = v[idx];
    double vx[4];
    if constexpr (THERMO == 2) {
        nhc = rshift(nhc, off);
#pragma unroll
        for (int k = 0; k < 4; ++k) vx[k] = nhc[(size_t)k * ndof + idx];
    }
    const double hdt = 0.5 * dt;
    if (do_close) {
        vi = fma(hdt, f, vi);
        if constexpr (THERMO == 1) {
            double z0, z1;
            philox_normal(seed, dof0 + idx, s_close, z0, z1);
            vi = c1 * vi + c2 * z1;
        } else if constexpr (THERMO == 2) {
            nhc_half(vi, vx, hdt, 1.0 / beta, Q);
        }
    }
    if (do_open) {
        if constexpr (THERMO == 1) {
            double z0, z1;
            philox_normal(seed, dof0 + idx, s_open, z0, z1);
            vi = c1 * vi + c2 * z0;
        } else if constexpr (THERMO == 2) {
            nhc_half(vi, vx, hdt, 1.0 / beta, Q);
        }
        vi = fma(hdt, f, vi);
        const double xn = fma(dt, vi, x[idx]);
        x[idx] = xn;
        if (!(fabs(xn) < INFINITY)) atomicOr(rshift(istatus, off), ST_NONFINITE);
    }
    v[idx] = vi;
    if constexpr (THERMO == 2) {
#pragma unroll
        for (int k = 0; k < 4; ++k) nhc[(size_t)k * ndof + idx] = vx[k];
    }
}

__global__ void __launch_bounds__(256) k_combine(double *__restrict__ out, const double *__restrict__ F,
                                                const double *__restrict__ Fex1, const double *__restrict__ FexP, size_t ndof,
                                                size_t slice, int P, int own_first, int own_last, size_t rs)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= ndof) return;
    const size_t off = (size_t)blockIdx.y * rs;
    F = rshift(F, off); Fex1 = rshift(Fex1, off); FexP = rshift(FexP, off);
    const size_t j = idx / slice, rem = idx - j * slice;
    double f = F[idx];
    if (j == 0 && own_first) f += Fex1[rem];
    if (j == (size_t)(P - 1) && own_last) f += FexP[rem];
    out[(size_t)blockIdx.y * ndof + idx] = f; // out: [B][P][N][d], contiguous
}

// ==========================================================================================
// Step 2 of the hot path: pair forces of one bead slice with Newton's third law,
//   F_l^j += (1/P) sum_{i != l} (2g/s^2) e^{-|r_l^j - r_i^j|^2/s^2} (r_l^j - r_i^j)      (Eq. 18)
// Particles are cut into tiles of 32.  Every unordered pair of tiles (I, J) is visited once through
// the cyclic scheme J = (I + m) mod NT, m = 1..H (H = (NT-1)/2; for even NT the last offset NT/2 is
// taken by I < NT/2 only).  A warp task owns row tile I and `ch` consecutive offsets m; lane t
// keeps particle i = 32 I + t and its force in registers.  Two column tiles are in flight at a time
// (two independent exp chains per lane).  At step k lane t meets column (t + k) mod 32 of each:
// positions come from shared memory (conflict free), the column's force accumulator travels from
// lane to lane (one shuffle rotation per step), so each Gaussian is evaluated once and used for both
// partners.  Tile results are added to F with FP64 atomics (F already holds the spring/trap forces).
// The last task of a row does the 32 x 32 diagonal tile the plain way.
// The Gaussian is exp_neg_tab256 (8 FP64 instructions; the 64-entry form with one more FMA measured 0.0811 against
// 0.0783 ms at cfg3).  Coordinates are pre-scaled by 1/s so that the exponent is -|dx'|^2; padding particles sit at
// +-1e150 and give e^-708 ~ 3e-308 (their forces are never written).
// grid (ceil(tasks/PAIR_WARPS), P, B), block PAIR_WARPS * 32; tasks = NT (nchunk + 1).
// ==========================================================================================
constexpr int PAIR_WARPS = 8;

// The pair potential v(r) of Eq. 18 (PAPER.md:142-144: "V" is generic; Eq. 20, :193, is the Gaussian instance) as a
// compile-time choice.  With r2 = |dx|^2 / s^2 (coordinates pre-scaled by 1/s) a potential gives
//   w  : force weight, F_i += coef * w * dx',  F_j -= the same     (coef carries the potential's constant factors)
//   u  : v(r) in units of the energy prefactor gE,   du : (v + r v'/2)(r) - v(r) in the same units (virial estimator)
//   POT 0  Gaussian       v = g exp(-r^2/s^2)      : w = u = e^{-r2},        du = -r2 e^{-r2};   coef = 2 g/(s P), gE = g
//   POT 1  soft Coulomb   v = g / sqrt(r^2 + s^2)  : w = (1+r2)^{-3/2}, u = (1+r2)^{-1/2}, du = -r2 w/2; coef = g/(s^2 P), gE = g/s
// Both are smooth at r = 0 with u(0) = 1, du(0) = 0 (the diagonal tile removes the self term analytically).
template <int POT> PIMD_DEV void pair_weight(double r2, const double *tab, double &w, double &u, double &du)
{
    if constexpr (POT == 0) {
        w = exp_neg_tab256(r2, tab);
        u = w;
        du = -w * fmin(r2, 708.0); // padding pairs have r2 ~ 1e300 and e = e^-708, not 0
    } else {
        const double rs = rsqrt(1.0 + r2);
        w = rs * rs * rs;
        u = rs;
        du = -0.5 * fmin(r2, 1e100) * w; // padding pairs: w = 0
    }
}

template <int D, bool EST, int POT>
PIMD_DEV void pair_term(const Vec<D> &ri, const double *sj, const double *tab, Vec<D> &fi, Vec<D> &fj, double &se, double &sea)
{
    Vec<D> dl;
#pragma unroll
    for (int c = 0; c < D; ++c) dl.v[c] = ri.v[c] - sj[c];
    double r2 = dl.v[0] * dl.v[0];
#pragma unroll
    for (int c = 1; c < D; ++c) r2 = fma(dl.v[c], dl.v[c], r2);
    double e, u, du;
    if constexpr (POT == 0 && !EST) e = exp_neg_tab256(r2, tab);
    else pair_weight<POT>(r2, tab, e, u, du);
#pragma unroll
    for (int c = 0; c < D; ++c) {
        fi.v[c] = fma(e, dl.v[c], fi.v[c]);
        fj.v[c] = fma(-e, dl.v[c], fj.v[c]);
    }
    if constexpr (EST) {
        se += u;
        sea += du;
    }
}

// 32 steps of lane t against NJ column tiles held twice over in shared memory (tl = tile + t*D, so
// that column (t + k) mod 32 is at the compile-time offset k*D); the column accumulators rotate.
template <int D, int NJ, bool EST, int POT>
PIMD_DEV void pair_sweep(const Vec<D> &ri, const double *tlA, const double *tlB, const double *tab, Vec<D> &fi, Vec<D> &fA,
                         Vec<D> &fB, double &se, double &sea, int nxt)
{
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        pair_term<D, EST, POT>(ri, tlA + k * D, tab, fi, fA, se, sea);
        if constexpr (NJ == 2) pair_term<D, EST, POT>(ri, tlB + k * D, tab, fi, fB, se, sea);
        if (k < 31) {
#pragma unroll
            for (int q = 0; q < D; ++q) {
                fA.v[q] = shfl_bcast(fA.v[q], nxt);
                if constexpr (NJ == 2) fB.v[q] = shfl_bcast(fB.v[q], nxt);
            }
        }
    }
}

template <int D, bool EST, int POT>
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_pair(const double *__restrict__ x, double *__restrict__ F, int N, int NT,
                                                         int nchunk, int ch, double inv_s, double coef /* 2 g / (s P) */,
                                                         double g, EstAccum *est, size_t rs)
{
    x = rshift(x, (size_t)blockIdx.z * rs); F = rshift(F, (size_t)blockIdx.z * rs);
    if constexpr (EST) est = rshift(est, (size_t)blockIdx.z * rs);
    __shared__ double tiles[PAIR_WARPS][2][64 * D];
    __shared__ double tab[256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int k = threadIdx.x; k < 256; k += PAIR_WARPS * 32) tab[k] = g_exp2_256[k];
    __syncthreads();
    const int task = blockIdx.x * PAIR_WARPS + warp;
    if (task >= NT * (nchunk + 1)) return; // warp-uniform; no block-wide barrier below
    const int I = task / (nchunk + 1), c = task - I * (nchunk + 1);
    const size_t sl = (size_t)blockIdx.y * N * D;
    const double *xs = x + sl;
    double *Fs = F + sl;
    double *tA = tiles[warp][0], *tB = tiles[warp][1];
    const double *tlA = tA + lane * D, *tlB = tB + lane * D;

    const int i = I * 32 + lane;
    const bool vi = i < N;
    Vec<D> ri, fi;
#pragma unroll
    for (int k = 0; k < D; ++k) { ri.v[k] = 1e150; fi.v[k] = 0.0; }
    if (vi) {
        ri = ldvec<D>(xs, i);
#pragma unroll
        for (int k = 0; k < D; ++k) ri.v[k] *= inv_s;
    }
    double se = 0.0, sea = 0.0;

    auto stage = [&](double *dst, int J) {
        const int jx = J * 32 + lane;
        Vec<D> p;
#pragma unroll
        for (int k = 0; k < D; ++k) p.v[k] = -1e150;
        if (jx < N) {
            p = ldvec<D>(xs, jx);
#pragma unroll
            for (int k = 0; k < D; ++k) p.v[k] *= inv_s;
        }
#pragma unroll
        for (int k = 0; k < D; ++k) { dst[lane * D + k] = p.v[k]; dst[(lane + 32) * D + k] = p.v[k]; }
    };
    auto flush = [&](int J, int col, const Vec<D> &f) {
        const int jx = J * 32 + col;
        if (jx < N) {
#pragma unroll
            for (int k = 0; k < D; ++k) atomicAdd(&Fs[(size_t)jx * D + k], coef * f.v[k]);
        }
    };
    const int nxt = (lane + 1) & 31, lastcol = (lane + 31) & 31;

    if (c == nchunk) {
        // diagonal tile: ordered pairs, the self term has dl = 0
        stage(tA, I);
        __syncwarp();
        Vec<D> dummy;
#pragma unroll
        for (int k = 0; k < D; ++k) dummy.v[k] = 0.0;
#pragma unroll 8
        for (int k = 0; k < 32; ++k) pair_term<D, EST, POT>(ri, tlA + k * D, tab, fi, dummy, se, sea);
        if constexpr (EST) {
            se = vi ? 0.5 * (se - 1.0) : 0.0;
            sea = vi ? 0.5 * sea : 0.0;
        }
    } else {
        const int H = (NT & 1) ? (NT - 1) / 2 : (NT / 2 - 1 + (I < NT / 2 ? 1 : 0));
        const int m0 = 1 + c * ch, m1 = min(m0 + ch - 1, H);
        int m = m0;
        for (; m + 1 <= m1; m += 2) {
            int JA = I + m, JB = I + m + 1;
            if (JA >= NT) JA -= NT;
            if (JB >= NT) JB -= NT;
            __syncwarp();
            stage(tA, JA);
            stage(tB, JB);
            __syncwarp();
            Vec<D> fA, fB;
#pragma unroll
            for (int k = 0; k < D; ++k) { fA.v[k] = 0.0; fB.v[k] = 0.0; }
            pair_sweep<D, 2, EST, POT>(ri, tlA, tlB, tab, fi, fA, fB, se, sea, nxt);
            flush(JA, lastcol, fA);
            flush(JB, lastcol, fB);
        }
        if (m <= m1) {
            int JA = I + m;
            if (JA >= NT) JA -= NT;
            __syncwarp();
            stage(tA, JA);
            __syncwarp();
            Vec<D> fA, fB;
#pragma unroll
            for (int k = 0; k < D; ++k) { fA.v[k] = 0.0; fB.v[k] = 0.0; }
            pair_sweep<D, 1, EST, POT>(ri, tlA, tlB, tab, fi, fA, fB, se, sea, nxt);
            flush(JA, lastcol, fA);
        }
    }
    if (vi) {
#pragma unroll
        for (int k = 0; k < D; ++k) atomicAdd(&Fs[(size_t)i * D + k], coef * fi.v[k]);
    }
    if constexpr (EST) {
        se = warp_sum(se);
        sea = warp_sum(sea);
        if (lane == 0) {
            atomicAdd(&est->upair, g * se);
            atomicAdd(&est->virpair, g * (se + sea));
        }
    }
}

// ==========================================================================================
// The same pair forces with TWO row particles per lane.  Tiles of 32 are paired into super-tiles of 64
// (S covers tiles 2S, 2S+1); the cyclic scheme runs over super-tiles.  Lane t keeps particles 64S + t and 64S + 32 + t
// and meets, at step k, column (t + k) mod 32 of both tiles of the partner super-tile: four potential evaluations per
// step (four independent exponential chains), every column position loaded once for two rows and every travelling
// column accumulator shuffled once for two contributions -- per pair half the LDS and SHFL traffic of k_pair, which was
// bound by the issue port (40 warp instructions per pair, 16 of them FP64; profiles/r1_measurements.md).
// The diagonal task of a super-tile does its two 32 x 32 diagonal tiles the plain way and the cross tile with
// Newton's third law.  grid (ceil(tasks/PAIR_WARPS), P, B), tasks = NS (nchunk + 1), NS = ceil(NT / 2).
// ==========================================================================================
template <int D, bool EST, int POT>
__global__ void __launch_bounds__(PAIR_WARPS * 32) k_pair2(const double *__restrict__ x, double *__restrict__ F, int N, int NS,
                                                          int nchunk, int ch, double inv_s, double coef, double g,
                                                          EstAccum *est, size_t rs)
{
    x = rshift(x, (size_t)blockIdx.z * rs); F = rshift(F, (size_t)blockIdx.z * rs);
    if constexpr (EST) est = rshift(est, (size_t)blockIdx.z * rs);
    __shared__ double tiles[PAIR_WARPS][2][64 * D];
    __shared__ double tab[256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int k = threadIdx.x; k < 256; k += PAIR_WARPS * 32) tab[k] = g_exp2_256[k];
    __syncthreads();
    const int task = blockIdx.x * PAIR_WARPS + warp;
    if (task >= NS * (nchunk + 1)) return; // warp-uniform; no block-wide barrier below
    const int S = task / (nchunk + 1), c = task - S * (nchunk + 1);
    const size_t sl = (size_t)blockIdx.y * N * D;
    const double *xs = x + sl;
    double *Fs = F + sl;
    double *tA = tiles[warp][0], *tB = tiles[warp][1];
    const double *tlA = tA + lane * D, *tlB = tB + lane * D;

    const int ia = S * 64 + lane, ib = ia + 32;
    const bool va = ia < N, vb = ib < N;
    Vec<D> ra, rb, fa, fb;
#pragma unroll
    for (int k = 0; k < D; ++k) { ra.v[k] = 1e150; rb.v[k] = 1e150; fa.v[k] = 0.0; fb.v[k] = 0.0; }
    if (va) {
        ra = ldvec<D>(xs, ia);
#pragma unroll
        for (int k = 0; k < D; ++k) ra.v[k] *= inv_s;
    }
    if (vb) {
        rb = ldvec<D>(xs, ib);
#pragma unroll
        for (int k = 0; k < D; ++k) rb.v[k] *= inv_s;
    }
    double se = 0.0, sea = 0.0;

    auto stage = [&](double *dst, int J) { // tile J of 32 particles, twice over (rotation by compile-time offsets)
        const int jx = J * 32 + lane;
        Vec<D> p;
#pragma unroll
        for (int k = 0; k < D; ++k) p.v[k] = -1e150;
        if (jx < N) {
            p = ldvec<D>(xs, jx);
#pragma unroll
            for (int k = 0; k < D; ++k) p.v[k] *= inv_s;
        }
#pragma unroll
        for (int k = 0; k < D; ++k) { dst[lane * D + k] = p.v[k]; dst[(lane + 32) * D + k] = p.v[k]; }
    };
    auto flush = [&](int J, int col, const Vec<D> &f) {
        const int jx = J * 32 + col;
        if (jx < N) {
#pragma unroll
            for (int k = 0; k < D; ++k) atomicAdd(&Fs[(size_t)jx * D + k], coef * f.v[k]);
        }
    };
    const int nxt = (lane + 1) & 31, lastcol = (lane + 31) & 31;
    Vec<D> zero;
#pragma unroll
    for (int k = 0; k < D; ++k) zero.v[k] = 0.0;

    if (c == nchunk) {
        // diagonal super-tile: tiles (2S, 2S) and (2S+1, 2S+1) as ordered pairs (the self term has dx = 0), tile pair
        // (2S, 2S+1) once with both partners
        stage(tA, 2 * S);
        stage(tB, 2 * S + 1);
        __syncwarp();
        double sd = 0.0, sda = 0.0;
        Vec<D> dummy = zero, fB = zero;
#pragma unroll 8
        for (int k = 0; k < 32; ++k) {
            pair_term<D, EST, POT>(ra, tlA + k * D, tab, fa, dummy, sd, sda);
            pair_term<D, EST, POT>(rb, tlB + k * D, tab, fb, dummy, sd, sda);
        }
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            pair_term<D, EST, POT>(ra, tlB + k * D, tab, fa, fB, se, sea);
            if (k < 31) {
#pragma unroll
                for (int q = 0; q < D; ++q) fB.v[q] = shfl_bcast(fB.v[q], nxt);
            }
        }
        flush(2 * S + 1, lastcol, fB);
        if constexpr (EST) {
            // ordered pairs count twice and include the self terms u(0) = 1 of the valid rows; pairs with a padding particle
            // carry u ~ e^-708 (Gaussian) or 0
            se += 0.5 * (sd - (va ? 1.0 : 0.0) - (vb ? 1.0 : 0.0));
            sea += 0.5 * sda;
        }
    } else {
        const int H = (NS & 1) ? (NS - 1) / 2 : (NS / 2 - 1 + (S < NS / 2 ? 1 : 0));
        const int m0 = 1 + c * ch, m1 = min(m0 + ch - 1, H);
        for (int m = m0; m <= m1; ++m) {
            int Sp = S + m;
            if (Sp >= NS) Sp -= NS;
            __syncwarp();
            stage(tA, 2 * Sp);
            stage(tB, 2 * Sp + 1);
            __syncwarp();
            Vec<D> fA = zero, fB = zero;
#pragma unroll
            for (int k = 0; k < 32; ++k) {
                pair_term<D, EST, POT>(ra, tlA + k * D, tab, fa, fA, se, sea);
                pair_term<D, EST, POT>(rb, tlA + k * D, tab, fb, fA, se, sea);
                pair_term<D, EST, POT>(ra, tlB + k * D, tab, fa, fB, se, sea);
                pair_term<D, EST, POT>(rb, tlB + k * D, tab, fb, fB, se, sea);
                if (k < 31) {
#pragma unroll
                    for (int q = 0; q < D; ++q) {
                        fA.v[q] = shfl_bcast(fA.v[q], nxt);
                        fB.v[q] = shfl_bcast(fB.v[q], nxt);
                    }
                }
            }
            flush(2 * Sp, lastcol, fA);
            flush(2 * Sp + 1, lastcol, fB);
        }
    }
    if (va) {
#pragma unroll
        for (int k = 0; k < D; ++k) atomicAdd(&Fs[(size_t)ia * D + k], coef * fa.v[k]);
    }
    if (vb) {
#pragma unroll
        for (int k = 0; k < D; ++k) atomicAdd(&Fs[(size_t)ib * D + k], coef * fb.v[k]);
    }
    if constexpr (EST) {
        se = warp_sum(se);
        sea = warp_sum(sea);
        if (lane == 0) {
            atomicAdd(&est->upair, g * se);
            atomicAdd(&est->virpair, g * (se + sea));
        }
    }
}

// ==========================================================================================
// Step 8: the estimators of one configuration from the sums the force kernels left behind (R9)
//   e_prim = P d N/(2 beta) - <E_c> + Ubar,  e_vir = Ubar + 1/2 sum r . grad Ubar,  Ubar = U/P
// and, when `accumulate` is set (pimd_run), their running sums and the running histograms.  One block per replica.
// Bead shards: `kin` and <E_c> are counted on rank 0 only, Ubar over the local slices, so the ranks' values add up.
// ==========================================================================================
struct EstSums {
    double n, sum_ep, sum_ev, last_ep, last_ev, pad[3];
};

__global__ void __launch_bounds__(256) k_estimate(int nspecies, const Scalars *scal, const EstAccum *est, EstSums *sums,
                                                 const double *hist, double *hist_acc, int nbins, const double *gr,
                                                 double *gr_acc, int nbins_gr, double kin, double ec_weight, double invP,
                                                 int accumulate, size_t rs)
{
    const size_t off = (size_t)blockIdx.x * rs;
    scal = rshift(scal, off); est = rshift(est, off); sums = rshift(sums, off);
    if (threadIdx.x == 0) {
        double ec = 0.0;
        for (int s = 0; s < nspecies; ++s) ec += scal[s].ec;
        const double ubar = est->utrap + est->upair * invP; // the trap term is accumulated already divided by P
        const double ep = ec_weight * (kin - ec) + ubar;
        const double ev = 2.0 * est->utrap + est->virpair * invP;
        sums->last_ep = ep;
        sums->last_ev = ev;
        if (accumulate) { sums->n += 1.0; sums->sum_ep += ep; sums->sum_ev += ev; }
    }
    if (accumulate) {
        hist = rshift(hist, off); hist_acc = rshift(hist_acc, off); gr = rshift(gr, off); gr_acc = rshift(gr_acc, off);
        for (int b = threadIdx.x; b < nbins; b += blockDim.x) hist_acc[b] += hist[b];
        for (int b = threadIdx.x; b < nbins_gr; b += blockDim.x) gr_acc[b] += gr[b];
    }
}

// ==========================================================================================
// Pair-distance histogram (pair-correlation estimator): counts of |r_l^j - r_i^j|, i < l, same bead
// index j (the pairs Eq. 18, couples), in nbins equal bins on [0, rmax); raw counts, normalisation by the
// caller.  Estimator steps only.  The distance is formed with separately rounded multiplies and adds (no FMA
// contraction), the order a plain C loop takes, so that the bin decision is the oracle's to the bit.
// grid (ceil(N/GR_TB), P, B), block GR_TB: thread = particle l, tiles of GR_TB partners through shared memory.
// ==========================================================================================
constexpr int GR_TB = 128;
constexpr int GR_MAXBINS = 4096;

template <int D>
__global__ void __launch_bounds__(GR_TB) k_gr(const double *__restrict__ x, int N, double *hist, int nbins, double rmax, size_t rs)
{
    __shared__ double tile[GR_TB * D];
    __shared__ unsigned int cnt[GR_MAXBINS];
    x = rshift(x, (size_t)blockIdx.z * rs); hist = rshift(hist, (size_t)blockIdx.z * rs);
    const double *xs = x + (size_t)blockIdx.y * N * D;
    for (int b = threadIdx.x; b < nbins; b += GR_TB) cnt[b] = 0u;
    const int l = blockIdx.x * GR_TB + threadIdx.x;
    Vec<D> r;
#pragma unroll
    for (int c = 0; c < D; ++c) r.v[c] = 0.0;
    if (l < N) r = ldvec<D>(xs, l);
    const int lmax = min(N, (blockIdx.x + 1) * GR_TB); // partners i < l only
    for (int t0 = 0; t0 < lmax; t0 += GR_TB) {
        __syncthreads();
        if (t0 + threadIdx.x < N) {
            const Vec<D> q = ldvec<D>(xs, t0 + threadIdx.x);
#pragma unroll
            for (int c = 0; c < D; ++c) tile[threadIdx.x * D + c] = q.v[c];
        }
        __syncthreads();
        const int kend = min(GR_TB, l - t0);
        for (int k = 0; k < kend; ++k) {
            double r2 = 0.0;
#pragma unroll
            for (int c = 0; c < D; ++c) {
                const double t = __dsub_rn(r.v[c], tile[k * D + c]);
                r2 = __dadd_rn(r2, __dmul_rn(t, t));
            }
            const double rr = sqrt(r2);
            if (l < N && rr < rmax) {
                int b = (int)(__dmul_rn(__ddiv_rn(rr, rmax), (double)nbins));
                if (b >= nbins) b = nbins - 1;
                atomicAdd(&cnt[b], 1u);
            }
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < nbins; b += GR_TB)
        if (cnt[b]) atomicAdd(&hist[b], (double)cnt[b]);
}

// ==========================================================================================
// Bead shards ("parallel computing ... with a large number of ... GPUs"; the
// per-slice pair term parallelises like classical MD).  A rank holds the contiguous slices [j0, j0 + Pl) of every ring.
// What leaves a rank per MD step is its boundary pack
//     [ first local slice : N d ][ last local slice : N d ][ partial E_int : N ]      (2 N d + N doubles, padded to even)
// (partial E_int = the springs between two local slices, Eq. 9); the all-gather of the packs gives every rank the halo
// slices of its ring neighbours, bead 1 (first slice of rank 0), bead P (last slice of the last rank) and, with the springs
// that cross a rank boundary added, E_int -- everything the exchange part (steps 3-6, run redundantly on every rank)
// and the local spring forces need.
// ==========================================================================================
template <int D>
__global__ void __launch_bounds__(128) k_shard_pack(const double *__restrict__ x, int N, int Pl, double ks, double *__restrict__ pack)
{
    const int l = blockIdx.x * 128 + threadIdx.x;
    if (l >= N) return;
    const size_t sl = (size_t)N * D;
    Vec<D> prev = ldvec<D>(x, l);
    stvec<D>(pack, l, prev);
    double acc = 0.0;
    for (int j = 1; j < Pl; ++j) {
        const Vec<D> cur = ldvec<D>(x + (size_t)j * sl, l);
        acc += dist2<D>(cur, prev);
        prev = cur;
    }
    stvec<D>(pack + sl, l, prev);
    pack[2 * sl + l] = 0.5 * ks * acc;
}

template <int D>
__global__ void __launch_bounds__(128) k_shard_eint(const double *__restrict__ gathered, int N, int world, size_t stride,
                                                   double ks, double *__restrict__ eint)
{
    const int l = blockIdx.x * 128 + threadIdx.x;
    if (l >= N) return;
    const size_t sl = (size_t)N * D;
    double e = 0.0, cross = 0.0;
    for (int r = 0; r < world; ++r) {
        e += gathered[r * stride + 2 * sl + l];
        if (r + 1 < world) cross += dist2<D>(ldvec<D>(gathered + (r + 1) * stride, l), ldvec<D>(gathered + r * stride + sl, l));
    }
    eint[l] = e + 0.5 * ks * cross;
}

// Pr of distinguishable particles (xi = 0): the identity
__global__ void __launch_bounds__(256) k_identity(int N, double *__restrict__ Pr)
{
    const int l = blockIdx.y, c0 = blockIdx.x * 1024 + threadIdx.x;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int lp = c0 + 256 * k;
        if (lp < N) __stcs(Pr + (size_t)l * N + lp, lp == l ? 1.0 : 0.0);
    }
}

__global__ void k_step_counter(unsigned long long *dstep, unsigned long long set, int add)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) *dstep = add ? *dstep + 1 : set;
}

// the device exponentials evaluated element-wise (parity tests): which = 0 exp_fast(x), 1 exp_tab(x),
// 2 exp_neg_tab64(x) = exp(-x), x >= 0
__global__ void __launch_bounds__(256) k_exp_selftest(const double *__restrict__ x, double *__restrict__ y, size_t n, int which)
{
    __shared__ double t32[32], t64[64], t256[256];
    if (threadIdx.x < 32) t32[threadIdx.x] = c_exp2_32[threadIdx.x];
    if (threadIdx.x < 64) t64[threadIdx.x] = c_exp2_64[threadIdx.x];
    t256[threadIdx.x] = g_exp2_256[threadIdx.x];
    __syncthreads();
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v = x[i];
    y[i] = which == 0 ? exp_fast(v) : (which == 1 ? exp_tab(v, t32) : (which == 2 ? exp_neg_tab64(v, t64) : exp_neg_tab256(v, t256)));
}

// FP64 FMA issue-rate probe: 8 independent chains per thread, register resident.
__global__ void __launch_bounds__(256) k_dfma_probe(double *out, int iters, double a, double b)
{
    double c0 = threadIdx.x, c1 = c0 + 1, c2 = c0 + 2, c3 = c0 + 3, c4 = c0 + 4, c5 = c0 + 5, c6 = c0 + 6, c7 = c0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            c0 = fma(c0, a, b); c1 = fma(c1, a, b); c2 = fma(c2, a, b); c3 = fma(c3, a, b);
            c4 = fma(c4, a, b); c5 = fma(c5, a, b); c6 = fma(c6, a, b); c7 = fma(c7, a, b);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((c0 + c1) + (c2 + c3)) + ((c4 + c5) + (c6 + c7));
}

} // namespace pimd
