// libpimd.so -- host side of the C ABI declared in include/pimd.h.
// Argument checking, workspace carving, stream fork/join and kernel launches only; every step of
// the hot path runs in the kernels of pimd_kernels.cuh.  There is no CPU fallback.
#include "../../include/pimd.h"
#include "pimd_kernels.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

using namespace pimd;

namespace {

thread_local char g_create_error[512] = "";

constexpr int BEAD_TB = 128;
constexpr int PREP_TB = 64;
constexpr int ASM_TB = 128;
constexpr int MAX_BINS = GR_MAXBINS;

// One exchange problem: the recursion of Eq. 6 / Eq. 11 over the particles [l0, l0 + N) of one species
// (several species = independent recursions over index ranges) with one parameter set
// (the sampling xi, or the second xi of pimd_reweight).  Pointers are those of replica 0.
struct ExchCtx {
    int N, l0, NB, nprep, nasm, nworkers;
    int sp; // species index: slot of this problem's gauge-misfit word in gflags (one launch = one species, all replicas)
    ExchPtrs p;
    Scalars *scal;
    double *ecpart;
    RepParams *rp;
    bool gauge_valid; // p.g / p.gs hold the (T, Zhat) of a completed evaluation of nearby positions
    int history;      // evaluations made along the current trajectory (pimd_set_state starts a new one): 2 allow extrapolation
};

} // namespace

struct pimd_s {
    int B, N, P, d;         // replicas, particles, bead slices held here (= Pg unless sharded), dimensions
    int Pg, j0, rank, world; // bead shards: global slice count, first local slice, rank of world
    bool sharded;
    double beta, omega, g, s, dt, gamma;
    int thermostat, pot;
    std::vector<double> *xi, *xi2;
    std::vector<uint64_t> *seed;
    bool any_neg[2], all_zero[2]; // per parameter set (0: sampling xi, 1: reweighting xi)
    uint64_t step;
    int nspecies, counts[PIMD_MAX_SPECIES];
    // derived
    double ks, kk;
    size_t ndof, slice;
    int look, look_spec, sms;
    int pair2_knob, pair_ch_knob; // PIMD_PAIR2 (-1: by size) and PIMD_PAIR_CH (0: by size), read once at creation
    // streams
    cudaStream_t s0, s1;
    cudaEvent_t ev_fork, ev_join;
    bool concurrent;
    // memory: [global region][replica 0][replica 1]...; pointers below are replica 0's
    unsigned char *ws;
    size_t ws_bytes, rstride;
    bool own_ws, carved;
    double *x, *v, *F, *nhc, *Fex1, *FexP, *Fexs1, *FexsP, *hist, *hist_acc, *gr, *gr_acc;
    ExchCtx ex[2][PIMD_MAX_SPECIES]; // [parameter set][species]
    RepParams *rp[2];
    Scalars *scal[2];
    EstAccum *est;
    EstSums *sums;
    int *istatus;
    // global region
    double *Fout, *gathered, *eint_tot, *pack, *Sarr, *Tarr;
    int *gflags;
    unsigned long long *fallbacks, *phase, *dstep;
    // one MD step (force evaluation, then close + open) captured as a CUDA graph on an internal stream
    cudaStream_t sg;
    cudaEvent_t ev_gin, ev_gout;
    cudaGraphExec_t gexec, gexec_est;
    bool use_graph, graph_failed, graph_conc;
    int graph_nbins, graph_nbins_gr;
    double graph_rmax, graph_rmax_gr;
    uint64_t graph_launches, graph_est_launches;
    // pinned host mirrors
    Scalars *h_scal;   // [B * MAX_SPECIES]
    EstSums *h_sums;   // [B]
    int *h_status;     // [B * (1 + 2 * MAX_SPECIES)]
    unsigned long long *h_diag;
    bool forces_valid;
    bool tables_valid; // the exchange tables of parameter set 0 belong to the current positions
    bool scalars_valid; // ... and k_finalize has run on them
    bool shard_imported;
    bool use_spec;     // PIMD_NOSPEC=1 turns the stale-gauge kernel off
    size_t spec_smem, chain_smem;
    int coop_max_blocks; // co-resident CTA limit of k_chain
    uint64_t launches;
    int nbins_gr;
    double rmax_gr;
    // per-kernel device timing (pimd_set_profiling)
    bool profiling;    // kernel launches bracketed by events
    bool phase_clock;  // ... and the chain CTA's clock64 instrumentation armed (PIMD_PROFILE_PHASES)
    std::vector<cudaEvent_t> *prof_ev; // pairs (start, stop)
    std::vector<int> *prof_slot;
    double prof_ms[PIMD_PROF_NSLOTS];
    uint64_t prof_n[PIMD_PROF_NSLOTS];
    char err[512];
};

namespace {

int fail(pimd_t h, int code, const char *fmt, ...)
{
    char *dst = h ? h->err : g_create_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

#define CU(call)                                                                                          \
    do {                                                                                                  \
        cudaError_t e__ = (call);                                                                         \
        if (e__ != cudaSuccess) return fail(h, PIMD_ECUDA, "%s: %s", #call, cudaGetErrorString(e__));     \
    } while (0)

// RAII bracket of one kernel launch with a pair of events on its stream (profiling mode only)
struct ProfScope {
    pimd_t h;
    cudaStream_t st;
    cudaEvent_t stop;
    ProfScope(pimd_t h_, int slot, cudaStream_t st_) : h(h_), st(st_), stop(nullptr)
    {
        h->launches++;
        if (!h->profiling) return;
        cudaEvent_t a = nullptr, b = nullptr;
        const size_t k = h->prof_slot->size();
        if (h->prof_ev->size() >= 2 * k + 2) { // recycled pair
            a = (*h->prof_ev)[2 * k];
            b = (*h->prof_ev)[2 * k + 1];
        } else {
            if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
            h->prof_ev->push_back(a);
            h->prof_ev->push_back(b);
        }
        h->prof_slot->push_back(slot);
        cudaEventRecord(a, st);
        stop = b;
    }
    ~ProfScope()
    {
        if (stop) cudaEventRecord(stop, st);
    }
};

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// doubles in a bead shard's boundary pack: first slice, last slice, partial E_int, padded to an even count so that the
// packs of all ranks stay 16-byte aligned in the gathered buffer (the slices are read as double2 for d = 2)
size_t pack_doubles_of(int N, int d) { return (2 * (size_t)N * d + (size_t)N + 1) / 2 * 2; }

// Carve the workspace; with base == nullptr only the sizes are computed.  Layout: the global region, then B replica
// regions of h->rstride bytes each with identical layout (kernels reach replica b through blockIdx * rstride).
size_t carve(pimd_t h, unsigned char *base)
{
    size_t off = 0;
    auto take = [&](size_t bytes) -> unsigned char * {
        unsigned char *p = base ? base + off : nullptr;
        off = align_up(off + bytes, 256);
        return p;
    };
    const size_t N = (size_t)h->N, D = (size_t)h->d, nd = h->ndof, B = (size_t)h->B;
    // ---- global region
    h->Fout = (double *)take(B * nd * 8);
    h->gflags = (int *)take(PIMD_MAX_SPECIES * 4);
    h->fallbacks = (unsigned long long *)take(8);
    h->phase = (unsigned long long *)take(16 * 8);
    h->dstep = (unsigned long long *)take(8);
    const size_t packn = pack_doubles_of(h->N, h->d);
    h->pack = (double *)take(h->sharded ? packn * 8 : 8);
    h->gathered = (double *)take(h->sharded ? (size_t)h->world * packn * 8 : 8);
    h->eint_tot = (double *)take(h->sharded ? N * 8 : 8);
    h->Sarr = (double *)take(N * 8);
    h->Tarr = (double *)take(N * 8);
    const size_t glob = off;
    // ---- replica 0
    h->x = (double *)take(nd * 8);
    h->v = (double *)take(nd * 8);
    h->F = (double *)take(nd * 8);
    h->nhc = (double *)take(h->thermostat == PIMD_THERMOSTAT_NHC ? nd * 8 * PIMD_NHC_LENGTH : 8);
    h->Fex1 = (double *)take(N * D * 8);
    h->FexP = (double *)take(N * D * 8);
    h->Fexs1 = (double *)take(N * D * 8); // exterior forces of the reweighting xi: computed, never used
    h->FexsP = (double *)take(N * D * 8);
    for (int set = 0; set < 2; ++set) {
        h->rp[set] = (RepParams *)take(sizeof(RepParams));
        h->scal[set] = (Scalars *)take(sizeof(Scalars) * PIMD_MAX_SPECIES);
        for (int sp = 0; sp < h->nspecies; ++sp) {
            ExchCtx &c = h->ex[set][sp];
            const size_t n = (size_t)c.N;
            for (int dir = 0; dir < 2; ++dir) {
                c.p.rho[dir] = (double *)take(n * D * 8);
                c.p.sig[dir] = (double *)take(n * D * 8);
                c.p.cc[dir] = (double *)take(n * 8);
                c.p.g[dir] = (double2 *)take((n + 1) * 16);
                c.p.gs[dir] = (double *)take((n + 1) * 8);
                c.p.gprev[dir] = (double2 *)take((n + 1) * 16);
                c.p.pan_m[dir] = (double *)take(n * 8);
                c.p.pan_s[dir] = (double *)take(n * 8);
                c.p.panel_ready[dir] = (int *)take((size_t)c.NB * 4);
                c.p.acc[dir] = (double *)take(n * (D + 2) * 8);
                c.p.pacc[dir] = (double *)take(n * (D + 1) * 8);
            }
            c.p.cols_ready = (int *)take(2 * 4);
            c.p.eint = (double *)take(n * 8);
            c.p.cnext = (double *)take(n * 8);
            c.p.cself = (double *)take(n * 8);
            c.p.pnext = (double *)take(n * 8);
            c.p.tpart = (double *)take((size_t)c.nprep * 2 * 8);
            c.p.rfin = (double2 *)take(2 * 16);
            c.p.rsgn = (double *)take(2 * 8);
            c.p.status = (int *)take(2 * 4);
            c.ecpart = (double *)take((size_t)c.nasm * 8);
            c.scal = h->scal[set] ? h->scal[set] + sp : nullptr;
            c.rp = h->rp[set];
        }
    }
    h->istatus = (int *)take(4);
    h->est = (EstAccum *)take(sizeof(EstAccum));
    h->sums = (EstSums *)take(sizeof(EstSums));
    h->hist = (double *)take((size_t)MAX_BINS * 8);
    h->hist_acc = (double *)take((size_t)MAX_BINS * 8);
    h->gr = (double *)take((size_t)MAX_BINS * 8);
    h->gr_acc = (double *)take((size_t)MAX_BINS * 8);
    h->rstride = off - glob;
    return glob + B * h->rstride;
}

int upload_params(pimd_t h, int set)
{
    std::vector<RepParams> rp((size_t)h->B);
    const std::vector<double> &xi = set ? *h->xi2 : *h->xi;
    h->any_neg[set] = false;
    h->all_zero[set] = true;
    for (int b = 0; b < h->B; ++b) {
        rp[b].xi = xi[b];
        rp[b].lambda = xi[b] != 0.0 ? std::log(std::fabs(xi[b])) : 0.0;
        rp[b].sx = xi[b] < 0.0 ? -1.0 : 1.0;
        rp[b].seed = (*h->seed)[b];
        if (xi[b] < 0.0) h->any_neg[set] = true;
        if (xi[b] != 0.0) h->all_zero[set] = false;
    }
    CU(cudaMemcpy2DAsync(h->rp[set], h->rstride, rp.data(), sizeof(RepParams), sizeof(RepParams), (size_t)h->B,
                         cudaMemcpyHostToDevice, h->s0));
    CU(cudaStreamSynchronize(h->s0)); // rp is a stack vector
    return PIMD_OK;
}

int ensure_ws(pimd_t h)
{
    if (h->carved) return PIMD_OK;
    const size_t need = carve(h, nullptr);
    if (!h->ws) {
        void *p = nullptr;
        cudaError_t e = cudaMalloc(&p, need);
        if (e != cudaSuccess) return fail(h, PIMD_ENOMEM, "cudaMalloc(%zu bytes): %s", need, cudaGetErrorString(e));
        h->ws = (unsigned char *)p;
        h->ws_bytes = need;
        h->own_ws = true;
    } else if (h->ws_bytes < need) {
        return fail(h, PIMD_ENOMEM, "workspace of %zu bytes is smaller than the %zu needed", h->ws_bytes, need);
    }
    carve(h, h->ws);
    CU(cudaMemsetAsync(h->ws, 0, need, h->s0));
    h->carved = true;
    int rc = upload_params(h, 0);
    if (rc) return rc;
    return upload_params(h, 1);
}

// species ranges -> exchange problems (both parameter sets); worker counts need the co-residency limit
int setup_species(pimd_t h)
{
    int l0 = 0;
    for (int sp = 0; sp < h->nspecies; ++sp) {
        for (int set = 0; set < 2; ++set) {
            ExchCtx &c = h->ex[set][sp];
            c.N = h->counts[sp];
            c.l0 = l0;
            c.sp = sp;
            c.NB = (c.N + 31) / 32;
            c.nprep = (c.N + PREP_TB - 1) / PREP_TB;
            c.nasm = (c.N + ASM_TB - 1) / ASM_TB;
            c.gauge_valid = false;
            c.history = 0;
            // Panel workers per direction.  A worker spins while it waits for columns and owns a whole SM, so only as many
            // as the panel work needs are launched: a worker needs about 480 NB cycles for its last row blocks and gets
            // nworkers x (one chain block, about 3000 cycles) for each, so NB/5 workers keep the panels ahead of the chain;
            // when the pair kernel dominates the step (g != 0 and P N large) the SMs are worth more there and NB/8 is enough.
            const int want = c.NB - h->look - 1;
            int cap = h->coop_max_blocks / (2 * h->B) - 1; // all replicas' CTAs must be co-resident
            int need = (h->g != 0.0 && (long long)h->P * h->N > 80000) ? (c.NB + 7) / 8 : (c.NB + 4) / 5;
            if (c.NB <= 80) need = (c.NB + 3) / 4; // a short chain leaves most SMs idle anyway: cfg3 7435 -> 7650 steps/s back to back with 14 instead of 10
            if (const char *e = std::getenv("PIMD_WORKERS")) {
                const int v = std::atoi(e);
                if (v >= 1) need = v;
            }
            if (need > cap) need = cap;
            // Row blocks beyond the look-ahead take their old columns from a panel worker, and the chain CTA waits for that
            // panel: with no room for even one worker per replica and direction the cooperative kernel would never finish.
            if (want > 0 && cap < 1)
                return fail(h, PIMD_EINVAL,
                            "a batch of %d replicas with %d particles in a species (more than %d) needs %d co-resident recursion CTAs "
                            "(chain + one panel worker, per direction and replica); the device holds %d: at most %d replicas",
                            h->B, c.N, 32 * (h->look + 1), 4 * h->B, h->coop_max_blocks, h->coop_max_blocks / 4);
            c.nworkers = want <= 0 ? 0 : std::max(0, std::min(want, need));
        }
        l0 += h->counts[sp];
    }
    return PIMD_OK;
}

template <int D> int setup_chain_attr(pimd_t h)
{
    const size_t smem = chain_smem_bytes_host<D>(h->look);
    h->chain_smem = smem;
    CU(cudaFuncSetAttribute(k_chain<D, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CU(cudaFuncSetAttribute(k_chain<D, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    h->spec_smem = chain_spec_smem_bytes_host<D>();
    if (h->spec_smem < smem) h->spec_smem = smem; // k_chain_spec holds the max-plus recursion as its safety net
    CU(cudaFuncSetAttribute(k_chain_spec<D, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->spec_smem));
    CU(cudaFuncSetAttribute(k_chain_spec<D, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->spec_smem));
    int nb = 0, dev = 0, sms = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_chain_spec<D, true>, CH_THREADS, h->spec_smem));
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    h->coop_max_blocks = nb * sms;
    h->sms = sms;
    if (h->coop_max_blocks < 2 * h->B)
        return fail(h, PIMD_EINVAL, "a batch of %d replicas needs %d co-resident recursion CTAs, the device holds %d", h->B, 2 * h->B,
                    h->coop_max_blocks);
    return PIMD_OK;
}

template <int D> int launch_bead(pimd_t h, cudaStream_t st, bool est, int nbins, double rmax)
{
    const dim3 grid((h->N + BEAD_TB - 1) / BEAD_TB, h->P, h->B), block(BEAD_TB);
    const double om2P = h->omega * h->omega / h->Pg;
    const size_t sl = h->slice, packn = pack_doubles_of(h->N, h->d);
    // bead shards: the ring neighbours' boundary slices come out of the gathered packs
    const double *halo_lo = (h->sharded && h->j0 > 0) ? h->gathered + (size_t)(h->rank - 1) * packn + sl : nullptr;
    const double *halo_hi = (h->sharded && h->j0 + h->P < h->Pg) ? h->gathered + (size_t)(h->rank + 1) * packn : nullptr;
    {
        // spring + trap forces (and the trap energy / histogram on estimator calls): F is written here
        ProfScope ps(h, PIMD_PROF_BEAD, st);
        if (est) k_bead<D, true, BEAD_TB><<<grid, block, 0, st>>>(h->x, h->F, h->N, h->P, h->ks, om2P, h->est, h->hist, nbins, rmax, halo_lo, halo_hi, h->rstride);
        else k_bead<D, false, BEAD_TB><<<grid, block, 0, st>>>(h->x, h->F, h->N, h->P, h->ks, om2P, h->est, h->hist, nbins, rmax, halo_lo, halo_hi, h->rstride);
    }
    CU(cudaGetLastError());
    if (h->g != 0.0) {
        // pair forces, added to F (Newton's third law, one potential evaluation per unordered pair)
        // From N = 1500 on: super-tiles of 64 particles, two row particles per lane (k_pair2: half the shared-memory and
        // shuffle traffic per pair; measured cfg3 0.0804 -> 0.0738 ms, cfg5b 1.199 -> 1.089 ms alone, but cfg4 (N = 1000)
        // 0.0398 -> 0.0422 and cfg2 0.0087 -> 0.0137: too few warps).  PIMD_PAIR2=0/1 forces one or the other.
        const bool two_rows = h->pair2_knob >= 0 ? h->pair2_knob != 0 : h->N >= 1500;
        const int NT = two_rows ? (h->N + 63) / 64 : (h->N + 31) / 32;
        const int hmax = (NT & 1) ? (NT - 1) / 2 : NT / 2;
        // tile offsets per task: small tasks balance the grid (one-row kernel: 1 is best up to N = 2500, 4 at N = 10000;
        // two-row kernel: 1 throughout, cfg5b 1.089 / 1.152 / 1.284 ms with 1 / 2 / 4); tuning knob PIMD_PAIR_CH
        int target = two_rows ? 1 : (NT <= 100 ? 1 : (NT <= 200 ? 2 : 4));
        if (h->pair_ch_knob > 0) target = h->pair_ch_knob;
        const int nchunk = hmax > 0 ? std::max(1, (hmax + target / 2) / target) : 0;
        const int ch = nchunk > 0 ? (hmax + nchunk - 1) / nchunk : 1;
        const long long tasks = (long long)NT * (nchunk + 1);
        const dim3 pgrid((unsigned)((tasks + PAIR_WARPS - 1) / PAIR_WARPS), h->P, h->B);
        // constant factors of the potential (pair_weight): force coefficient and energy prefactor
        const double coef = h->pot == 0 ? 2.0 * h->g / (h->s * h->Pg) : h->g / (h->s * h->s * h->Pg);
        const double gE = h->pot == 0 ? h->g : h->g / h->s;
        ProfScope ps(h, PIMD_PROF_PAIR, st);
#define LP(E, POT)                                                                                                                    \
    do {                                                                                                                              \
        if (two_rows) k_pair2<D, E, POT><<<pgrid, PAIR_WARPS * 32, 0, st>>>(h->x, h->F, h->N, NT, nchunk, ch, 1.0 / h->s, coef, gE, h->est, h->rstride); \
        else k_pair<D, E, POT><<<pgrid, PAIR_WARPS * 32, 0, st>>>(h->x, h->F, h->N, NT, nchunk, ch, 1.0 / h->s, coef, gE, h->est, h->rstride);           \
    } while (0)
        if (h->pot == 0) { if (est) LP(true, 0); else LP(false, 0); }
        else { if (est) LP(true, 1); else LP(false, 1); }
#undef LP
    }
    CU(cudaGetLastError());
    if (est && h->nbins_gr > 0) {
        const dim3 ggrid((h->N + GR_TB - 1) / GR_TB, h->P, h->B);
        ProfScope ps(h, PIMD_PROF_GR, st);
        k_gr<D><<<ggrid, GR_TB, 0, st>>>(h->x, h->N, h->gr, h->nbins_gr, h->rmax_gr, h->rstride);
        CU(cudaGetLastError());
    }
    return PIMD_OK;
}

template <int D> int launch_prep(pimd_t h, ExchCtx &c, cudaStream_t st)
{
    const size_t sl = h->slice, packn = pack_doubles_of(h->N, h->d), lo = (size_t)c.l0 * D;
    const double *x = h->x + lo, *x1 = h->x + lo, *xP = h->x + (size_t)(h->P - 1) * sl + lo, *ein = nullptr;
    if (h->sharded) { // bead 1 = first slice of rank 0, bead P = last slice of the last rank, E_int summed over the ranks
        x = nullptr;
        x1 = h->gathered + lo;
        xP = h->gathered + (size_t)(h->world - 1) * packn + sl + lo;
        ein = h->eint_tot + c.l0;
    }
    {
        ProfScope ps(h, PIMD_PROF_PREP, st);
        k_prep<D, PREP_TB><<<dim3(c.nprep, h->B), PREP_TB * PREP_SPLIT, 0, st>>>(x, x1, xP, ein, sl, c.N, h->P, c.NB, h->ks, h->kk, c.p, c.rp,
                                                                               h->gflags + c.sp, c.history >= 2 ? 1 : 0, h->rstride);
    }
    CU(cudaGetLastError());
    return PIMD_OK;
}

template <int D> int launch_exchange(pimd_t h, ExchCtx &c, int set, cudaStream_t st, bool scalars)
{
    const bool sgn = h->any_neg[set];
    const size_t lo = (size_t)c.l0 * D;
    double *const Fex1 = set ? h->Fexs1 : h->Fex1, *const FexP = set ? h->FexsP : h->FexP;
    if (h->all_zero[set]) {
        {
            ProfScope ps(h, PIMD_PROF_ASSEMBLE, st);
            k_exch_xi0<D, ASM_TB><<<dim3(c.nasm, h->B), ASM_TB, 0, st>>>(c.N, h->ks, c.p, Fex1 + lo, FexP + lo, c.ecpart, h->rstride);
        }
        CU(cudaGetLastError());
    } else {
        ChainArgs a;
        a.N = c.N; a.NB = c.NB; a.look = h->look; a.nworkers = c.nworkers;
        a.kk = h->kk; a.p = c.p; a.rp = c.rp; a.rs = h->rstride;
        a.phase = h->phase_clock ? h->phase : nullptr;
        a.look_fb = h->look;
        a.ks = h->ks; a.Fex1 = Fex1 + lo; a.FexP = FexP + lo; a.ecpart = c.ecpart;
        a.gauge_misfit = h->gflags + c.sp; // a species that rejects its gauge must not make the later ones redo theirs
        a.fallbacks = h->fallbacks;
        void *args[] = {&a};
        const dim3 grid(1 + c.nworkers, 2, h->B), block(CH_THREADS);
        if (c.gauge_valid && h->use_spec) {
            // the previous evaluation's gauge is at hand: linear pass only; the kernel redoes the recursion with a
            // fresh max-plus gauge itself (after a grid barrier) if the gauge turned out not to fit
            const void *fs = sgn ? (const void *)k_chain_spec<D, true> : (const void *)k_chain_spec<D, false>;
            a.look = h->look_spec; // the workers need one more block of head start when the chain runs this fast
            ProfScope ps(h, PIMD_PROF_CHAIN, st);
            CU(cudaLaunchCooperativeKernel(fs, grid, block, args, h->spec_smem, st));
        } else {
            const void *fn = sgn ? (const void *)k_chain<D, true> : (const void *)k_chain<D, false>;
            ProfScope ps(h, PIMD_PROF_CHAIN, st);
            CU(cudaLaunchCooperativeKernel(fn, grid, block, args, h->chain_smem, st));
        }
        c.gauge_valid = true;
        c.history++;
        // the force band (LOOK + 1 newest column blocks per row block) and the assembly of the exterior forces run as
        // the tail of the recursion kernel (exchange_tail)
    }
    if (scalars) {
        {
            ProfScope ps(h, PIMD_PROF_FINALIZE, st);
            k_finalize<256><<<h->B, 256, 0, st>>>(c.N, c.nprep, c.nasm, h->beta, c.rp, std::lgamma((double)c.N + 1.0), c.p, c.ecpart, c.scal,
                                                  h->rstride);
        }
        CU(cudaGetLastError());
    }
    return PIMD_OK;
}

int prep_d(pimd_t h, ExchCtx &c, cudaStream_t st)
{
    switch (h->d) {
    case 1: return launch_prep<1>(h, c, st);
    case 2: return launch_prep<2>(h, c, st);
    default: return launch_prep<3>(h, c, st);
    }
}
int exchange_d(pimd_t h, ExchCtx &c, int set, cudaStream_t st, bool scalars)
{
    switch (h->d) {
    case 1: return launch_exchange<1>(h, c, set, st, scalars);
    case 2: return launch_exchange<2>(h, c, set, st, scalars);
    default: return launch_exchange<3>(h, c, set, st, scalars);
    }
}
int bead_d(pimd_t h, cudaStream_t st, bool est, int nbins, double rmax)
{
    switch (h->d) {
    case 1: return launch_bead<1>(h, st, est, nbins, rmax);
    case 2: return launch_bead<2>(h, st, est, nbins, rmax);
    default: return launch_bead<3>(h, st, est, nbins, rmax);
    }
}

// the estimators of the evaluation just made (k_estimate), optionally added to the running sums
int launch_estimate(pimd_t h, int nbins, bool accumulate)
{
    const double kin = (double)h->Pg * h->d * h->N / (2.0 * h->beta);
    const double ecw = (!h->sharded || h->rank == 0) ? 1.0 : 0.0;
    ProfScope ps(h, PIMD_PROF_FINALIZE, h->s0);
    k_estimate<<<h->B, 256, 0, h->s0>>>(h->nspecies, h->scal[0], h->est, h->sums, h->hist, h->hist_acc, nbins, h->gr, h->gr_acc,
                                        h->nbins_gr, kin, ecw, 1.0 / h->Pg, accumulate ? 1 : 0, h->rstride);
    CU(cudaGetLastError());
    return PIMD_OK;
}

// one force evaluation.  The exchange part stays on the main stream (k_prep, then the latency-bound
// k_chain, which must get its SMs first), the bead part (spring/trap/pair) is forked onto the helper
// stream after k_prep and fills the remaining SMs; joined before returning (in stream order).
int eval_forces(pimd_t h, bool scalars, bool est, int nbins, double rmax)
{
    int rc = ensure_ws(h);
    if (rc) return rc;
    if (h->sharded && !h->shard_imported) return fail(h, PIMD_EINVAL, "bead shard: no boundary data imported for the current positions");
    if (est) {
        CU(cudaMemset2DAsync(h->est, h->rstride, 0, sizeof(EstAccum), (size_t)h->B, h->s0));
        if (nbins > 0) CU(cudaMemset2DAsync(h->hist, h->rstride, 0, (size_t)nbins * 8, (size_t)h->B, h->s0));
        if (h->nbins_gr > 0) CU(cudaMemset2DAsync(h->gr, h->rstride, 0, (size_t)h->nbins_gr * 8, (size_t)h->B, h->s0));
    }
    cudaStream_t sb = h->concurrent ? h->s1 : h->s0;
    for (int sp = 0; sp < h->nspecies; ++sp) {
        rc = prep_d(h, h->ex[0][sp], h->s0);
        if (rc) return rc;
    }
    if (h->concurrent) {
        CU(cudaEventRecord(h->ev_fork, h->s0));
        CU(cudaStreamWaitEvent(h->s1, h->ev_fork, 0));
    }
    for (int sp = 0; sp < h->nspecies; ++sp) {
        rc = exchange_d(h, h->ex[0][sp], 0, h->s0, scalars || est);
        if (rc) return rc;
    }
    rc = bead_d(h, sb, est, nbins, rmax);
    if (rc) return rc;
    if (h->concurrent) {
        CU(cudaEventRecord(h->ev_join, h->s1));
        CU(cudaStreamWaitEvent(h->s0, h->ev_join, 0));
    }
    h->forces_valid = true;
    h->tables_valid = true;
    h->scalars_valid = scalars || est;
    return PIMD_OK;
}

int launch_integrate(pimd_t h, bool do_close, bool do_open, uint64_t step_close, uint64_t step_open, bool device_counter = false)
{
    const unsigned long long *dstep = device_counter ? h->dstep : nullptr;
    const double c1 = std::exp(-h->gamma * h->dt * 0.5);
    const double c2 = std::sqrt((1.0 - c1 * c1) / h->beta);
    const double Q = h->beta / (double)h->Pg;
    const dim3 grid((unsigned)((h->ndof + 255) / 256), h->B);
    const int own_first = (!h->sharded || h->j0 == 0) ? 1 : 0, own_last = (!h->sharded || h->j0 + h->P == h->Pg) ? 1 : 0;
    const size_t dof0 = (size_t)h->j0 * h->slice;
#define LI(T) \
    k_integrate<T><<<grid, 256, 0, h->s0>>>(h->x, h->v, h->F, h->Fex1, h->FexP, h->nhc, h->ndof, h->slice, h->P, h->dt, c1, c2, \
                                            h->beta, Q, h->rp[0], step_close, step_open, do_close ? 1 : 0, do_open ? 1 : 0,     \
                                            h->istatus, dstep, own_first, own_last, dof0, h->rstride)
    {
        ProfScope ps(h, PIMD_PROF_INTEGRATE, h->s0);
        if (h->thermostat == PIMD_THERMOSTAT_LANGEVIN) LI(1);
        else if (h->thermostat == PIMD_THERMOSTAT_NHC) LI(2);
        else LI(0);
    }
#undef LI
    CU(cudaGetLastError());
    if (do_open) h->shard_imported = false; // positions moved: the boundary data is stale
    return PIMD_OK;
}

// status words of the last evaluation (every replica, every species) and of the integrator; synchronises
int read_status(pimd_t h)
{
    const int B = h->B, S = h->nspecies;
    CU(cudaMemcpy2DAsync(h->h_status, 4, h->istatus, h->rstride, 4, (size_t)B, cudaMemcpyDeviceToHost, h->s0));
    for (int sp = 0; sp < S; ++sp)
        CU(cudaMemcpy2DAsync(h->h_status + (size_t)B * (1 + sp), 4, h->ex[0][sp].p.status, h->rstride, 4, (size_t)B, cudaMemcpyDeviceToHost, h->s0));
    CU(cudaStreamSynchronize(h->s0));
    int st = 0;
    for (int k = 0; k < B * (1 + S); ++k) st |= h->h_status[k];
    if (st & ST_NONFINITE) return fail(h, PIMD_ENUMERIC, "non-finite state or potential");
    if (st & ST_NODE) return fail(h, PIMD_ENUMERIC, "e^{-beta V} summed to zero (node of the xi<0 weight)");
    return PIMD_OK;
}

bool finite_all(std::initializer_list<double> v)
{
    for (double a : v)
        if (!std::isfinite(a)) return false;
    return true;
}

void drop_graphs(pimd_t h)
{
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    if (h->gexec_est) { cudaGraphExecDestroy(h->gexec_est); h->gexec_est = nullptr; }
}

// Capture "force evaluation ; [estimators] ; close step s + open step s+1 ; counter += 1" once, on an internal stream
// (the caller's stream may be the legacy default stream, which cannot be captured).  Any failure (e.g. a driver that
// cannot put a cooperative launch into a graph) switches the feature off for this handle; nothing else depends on it.
int capture_step(pimd_t h, bool est, int nbins, double rmax, cudaGraphExec_t *out, uint64_t *nlaunch)
{
    if (h->graph_failed) return PIMD_ECUDA;
    cudaStream_t user = h->s0;
    const uint64_t l0 = h->launches;
    const bool fv = h->forces_valid, tv = h->tables_valid, sv = h->scalars_valid;
    cudaGraph_t graph = nullptr;
    int rc = PIMD_OK;
    if (cudaStreamBeginCapture(h->sg, cudaStreamCaptureModeRelaxed) != cudaSuccess) rc = PIMD_ECUDA;
    if (rc == PIMD_OK) {
        h->s0 = h->sg;
        rc = eval_forces(h, false, est, nbins, rmax);
        if (rc == PIMD_OK && est) rc = launch_estimate(h, nbins, true);
        if (rc == PIMD_OK) rc = launch_integrate(h, true, true, 0, 0, true);
        if (rc == PIMD_OK) {
            k_step_counter<<<1, 32, 0, h->sg>>>(h->dstep, 0ull, 1);
            h->launches++;
            if (cudaGetLastError() != cudaSuccess) rc = PIMD_ECUDA;
        }
        h->s0 = user;
        if (cudaStreamEndCapture(h->sg, &graph) != cudaSuccess || !graph) rc = PIMD_ECUDA;
    }
    if (rc == PIMD_OK && cudaGraphInstantiate(out, graph, 0) != cudaSuccess) rc = PIMD_ECUDA;
    if (graph) cudaGraphDestroy(graph);
    *nlaunch = h->launches - l0;
    h->launches = l0;
    h->forces_valid = fv;
    h->tables_valid = tv;
    h->scalars_valid = sv;
    if (rc != PIMD_OK) {
        cudaGetLastError();
        *out = nullptr;
        h->graph_failed = true;
        return PIMD_ECUDA;
    }
    return PIMD_OK;
}

int ensure_graphs(pimd_t h, bool need_est, int nbins, double rmax)
{
    if (h->graph_conc != h->concurrent) drop_graphs(h);
    if (h->gexec_est && (h->graph_nbins != nbins || h->graph_rmax != rmax || h->graph_nbins_gr != h->nbins_gr || h->graph_rmax_gr != h->rmax_gr)) {
        cudaGraphExecDestroy(h->gexec_est);
        h->gexec_est = nullptr;
    }
    h->graph_conc = h->concurrent;
    if (!h->gexec) {
        int rc = capture_step(h, false, 0, 0.0, &h->gexec, &h->graph_launches);
        if (rc) return rc;
    }
    if (need_est && !h->gexec_est) {
        int rc = capture_step(h, true, nbins, rmax, &h->gexec_est, &h->graph_est_launches);
        if (rc) return rc;
        h->graph_nbins = nbins; h->graph_rmax = rmax; h->graph_nbins_gr = h->nbins_gr; h->graph_rmax_gr = h->rmax_gr;
    }
    return PIMD_OK;
}

// nsteps MD steps; with est_every > 0 the force evaluation of every step whose (absolute) number is a multiple of
// est_every runs in estimator mode and its estimators are added to the running sums
int run_steps(pimd_t h, int nsteps, int est_every, int nbins, double rmax)
{
    if (nsteps == 0) return PIMD_OK;
    int rc = ensure_ws(h);
    if (rc) return rc;
    if (h->sharded) return fail(h, PIMD_EINVAL, "bead shard: advance with pimd_shard_begin_step / pimd_shard_end_step");
    if (!h->forces_valid) {
        rc = eval_forces(h, false, false, 0, 0.0);
        if (rc) return rc;
    }
    auto is_est = [&](uint64_t step_done) { return est_every > 0 && step_done % (uint64_t)est_every == 0; };
    // open step s ; forces ; [close s + open s+1] ; forces ; ... ; close last
    rc = launch_integrate(h, false, true, 0, h->step);
    if (rc) return rc;
    // Steps are launched one by one until the stale-gauge kernel with extrapolation is what a step runs (two
    // evaluations along this trajectory); from then on all but the last step replay the captured graphs, the step
    // counter of the noise living on the device meanwhile.
    auto graph_ready = [&]() {
        if (!h->use_graph || h->profiling) return false;
        for (int sp = 0; sp < h->nspecies; ++sp)
            if (!h->all_zero[0] && !(h->ex[0][sp].gauge_valid && h->ex[0][sp].history >= 2)) return false;
        return true;
    };
    int it = 0;
    while (it < nsteps) {
        if (nsteps - it >= 3 && graph_ready() && ensure_graphs(h, est_every > 0, nbins, rmax) == PIMD_OK) {
            k_step_counter<<<1, 32, 0, h->s0>>>(h->dstep, (unsigned long long)h->step, 0);
            CU(cudaGetLastError());
            CU(cudaEventRecord(h->ev_gin, h->s0));
            CU(cudaStreamWaitEvent(h->sg, h->ev_gin, 0));
            for (; it < nsteps - 1; ++it) {
                const bool e = is_est(h->step + 1);
                CU(cudaGraphLaunch(e ? h->gexec_est : h->gexec, h->sg));
                h->launches += e ? h->graph_est_launches : h->graph_launches;
                h->step++;
            }
            CU(cudaEventRecord(h->ev_gout, h->sg));
            CU(cudaStreamWaitEvent(h->s0, h->ev_gout, 0));
            continue;
        }
        const bool e = is_est(h->step + 1);
        rc = eval_forces(h, false, e, nbins, rmax);
        if (rc == PIMD_OK && e) rc = launch_estimate(h, nbins, true);
        if (rc) return rc;
        const bool last = it == nsteps - 1;
        rc = launch_integrate(h, true, !last, h->step, h->step + 1);
        if (rc) return rc;
        h->step++;
        ++it;
    }
    return PIMD_OK; // the flags eval_forces set for the last step hold: F, the tables belong to the final positions
}

} // namespace

template <int D> static int cycle_energies_impl(pimd_t h, double *e_dev)
{
    ExchCtx &c = h->ex[0][0];
    int rc = launch_prep<D>(h, c, h->s0); // E_int, C(l,l+1), bead-1 / bead-P slices of the current positions
    if (rc) return rc;
    k_prefix_st<<<1, 1024, 0, h->s0>>>(c.N, h->beta, c.p.eint, c.p.cnext, h->Sarr, h->Tarr);
    CU(cudaGetLastError());
    const dim3 grid((c.N + 1023) / 1024, c.N);
    {
        ProfScope ps(h, PIMD_PROF_EMAT, h->s0);
        k_emat<D><<<grid, 256, 0, h->s0>>>(c.N, h->ks, c.p.rho[0], c.p.sig[0], h->Sarr, h->Tarr, e_dev);
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(h->s0));
    h->tables_valid = false; // k_prep cleared the accumulators of the last evaluation
    h->scalars_valid = false;
    return PIMD_OK;
}

template <int D> static int prmat_impl(pimd_t h, double *pr_dev)
{
    ExchCtx &c = h->ex[0][0];
    const int N = c.N;
    const dim3 grid((N + 1023) / 1024, N), gridp((N + 256 * PRMAT_COLS - 1) / (256 * PRMAT_COLS), (N + PRMAT_ROWS - 1) / PRMAT_ROWS);
    ProfScope ps(h, PIMD_PROF_PRMAT, h->s0);
    if (h->all_zero[0]) k_identity<<<grid, 256, 0, h->s0>>>(N, pr_dev);
    else if (h->any_neg[0]) k_prmat<D, true><<<gridp, 256, 0, h->s0>>>(N, h->kk, c.p, pr_dev);
    else k_prmat<D, false><<<gridp, 256, 0, h->s0>>>(N, h->kk, c.p, pr_dev);
    return PIMD_OK;
}

static int create_impl(pimd_t *out, int B, bool shard, int rank, int world, int N, int P, int d, double beta, double omega, double g, double s,
                       const double *xi, double dt, int thermostat, const uint64_t *seed)
{
    pimd_t h = nullptr;
    if (!out) return fail(nullptr, PIMD_EINVAL, "out is NULL");
    *out = nullptr;
    if (N < 1 || P < 2 || d < 1 || d > 3) return fail(nullptr, PIMD_EINVAL, "need N >= 1, P >= 2, d in {1,2,3} (got N=%d P=%d d=%d)", N, P, d);
    if (B < 1 || !xi || !seed) return fail(nullptr, PIMD_EINVAL, "need B >= 1 replicas with xi[B] and seed[B]");
    if (world < 1 || rank < 0 || rank >= world || world > P) return fail(nullptr, PIMD_EINVAL, "need 0 <= rank < world <= P (got rank=%d world=%d P=%d)", rank, world, P);
    if (shard && B != 1) return fail(nullptr, PIMD_EINVAL, "bead shards hold one replica");
    if (!finite_all({beta, omega, g, s, dt}) || !(beta > 0) || !(s > 0) || !(dt > 0) || omega < 0)
        return fail(nullptr, PIMD_EINVAL, "need finite arguments with beta > 0, s > 0, dt > 0, omega >= 0");
    bool any0 = false, anynz = false;
    for (int b = 0; b < B; ++b) {
        if (!std::isfinite(xi[b])) return fail(nullptr, PIMD_EINVAL, "xi must be finite");
        if (xi[b] == 0.0) any0 = true; else anynz = true;
    }
    if (any0 && anynz) return fail(nullptr, PIMD_EINVAL, "a batch is either all xi = 0 (distinguishable particles) or all xi != 0");
    if (thermostat < 0 || thermostat > 2) return fail(nullptr, PIMD_EINVAL, "thermostat must be 0, 1 or 2");
    if ((double)N * P * d > 2.0e9) return fail(nullptr, PIMD_EINVAL, "N*P*d too large");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1)
        return fail(nullptr, PIMD_ECUDA, "no CUDA device (%s); libpimd has no CPU fallback", e != cudaSuccess ? cudaGetErrorString(e) : "count 0");
    h = new (std::nothrow) pimd_s();
    if (!h) return fail(nullptr, PIMD_ENOMEM, "host allocation failed");
    std::memset(h, 0, sizeof(*h));
    h->B = B; h->N = N; h->d = d;
    h->Pg = P; h->rank = rank; h->world = world; h->sharded = shard; // world = 1 is a valid (degenerate) shard
    // bead shards: rank r holds the slices [floor(P r / world), floor(P (r+1) / world))
    h->j0 = (int)((long long)P * rank / world);
    h->P = (int)((long long)P * (rank + 1) / world) - h->j0;
    h->beta = beta; h->omega = omega; h->g = g; h->s = s; h->dt = dt; h->gamma = 1.0;
    h->thermostat = thermostat; h->step = 0; h->pot = PIMD_PAIR_GAUSSIAN;
    h->xi = new std::vector<double>(xi, xi + B);
    h->xi2 = new std::vector<double>(xi, xi + B);
    h->seed = new std::vector<uint64_t>(seed, seed + B);
    h->ks = (double)P / (beta * beta);          // m omega_P^2, omega_P = sqrt(P)/(beta hbar)
    h->kk = (double)P / (2.0 * beta);           // beta k_s / 2
    h->slice = (size_t)N * d;
    h->ndof = h->slice * h->P;
    h->nspecies = 1;
    h->counts[0] = N;
    h->look = 3;      // column blocks kept inside the chain CTA: the same for the max-plus and the stale-gauge recursion,
    h->look_spec = 3; // because the force pass covers exactly those blocks and the workers' panels everything older
    if (const char *e2 = std::getenv("PIMD_LOOK")) { // tuning knob: column blocks kept inside the chain CTA
        const int v = std::atoi(e2);
        if (v >= 1 && v <= CH_MAXLOOK) h->look = h->look_spec = v;
    }
    h->pair2_knob = -1;
    if (const char *e2 = std::getenv("PIMD_PAIR2")) h->pair2_knob = std::atoi(e2) != 0 ? 1 : 0;
    h->pair_ch_knob = 0;
    if (const char *e2 = std::getenv("PIMD_PAIR_CH")) { const int v = std::atoi(e2); if (v >= 1 && v <= 64) h->pair_ch_knob = v; }
    h->concurrent = true;
    h->use_graph = !(std::getenv("PIMD_GRAPH") && std::atoi(std::getenv("PIMD_GRAPH")) == 0);
    h->use_spec = !(std::getenv("PIMD_NOSPEC") && std::atoi(std::getenv("PIMD_NOSPEC")) != 0);
    h->prof_ev = new std::vector<cudaEvent_t>();
    h->prof_slot = new std::vector<int>();
    int rc = PIMD_OK;
    auto bail = [&](int code) { std::snprintf(g_create_error, 512, "%s", h->err); pimd_destroy(h); return code; };
    switch (d) {
    case 1: rc = setup_chain_attr<1>(h); break;
    case 2: rc = setup_chain_attr<2>(h); break;
    default: rc = setup_chain_attr<3>(h); break;
    }
    if (rc) return bail(rc);
    rc = setup_species(h);
    if (rc) return bail(rc);
    const size_t nst = (size_t)B * (1 + 2 * PIMD_MAX_SPECIES);
    if (cudaStreamCreateWithFlags(&h->s1, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&h->sg, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_gin, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_gout, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_scal, sizeof(Scalars) * (size_t)B * PIMD_MAX_SPECIES) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_sums, sizeof(EstSums) * (size_t)B) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_diag, 16) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_status, nst * sizeof(int)) != cudaSuccess)
        return bail(fail(h, PIMD_ECUDA, "stream/event/pinned allocation failed: %s", cudaGetErrorString(cudaGetLastError())));
    *out = h;
    return PIMD_OK;
}

extern "C" {

const char *pimd_version(void) { return "pimd-b200 0.2 (sm_100a)"; }

const char *pimd_last_error(pimd_t h) { return h ? h->err : g_create_error; }

int pimd_create(pimd_t *out, int N, int P, int d, double beta, double omega, double g, double s, double xi, double dt,
                int thermostat, uint64_t seed)
{
    return create_impl(out, 1, false, 0, 1, N, P, d, beta, omega, g, s, &xi, dt, thermostat, &seed);
}

int pimd_create_batch(pimd_t *out, int B, int N, int P, int d, double beta, double omega, double g, double s, const double *xi,
                      double dt, int thermostat, const uint64_t *seed)
{
    return create_impl(out, B, false, 0, 1, N, P, d, beta, omega, g, s, xi, dt, thermostat, seed);
}

int pimd_create_sharded(pimd_t *out, int rank, int world, int N, int P, int d, double beta, double omega, double g, double s,
                        double xi, double dt, int thermostat, uint64_t seed)
{
    return create_impl(out, 1, true, rank, world, N, P, d, beta, omega, g, s, &xi, dt, thermostat, &seed);
}

int pimd_destroy(pimd_t h)
{
    if (!h) return PIMD_OK;
    if (h->s0 || h->s1) cudaDeviceSynchronize();
    if (h->own_ws && h->ws) cudaFree(h->ws);
    drop_graphs(h);
    if (h->sg) cudaStreamDestroy(h->sg);
    if (h->ev_gin) cudaEventDestroy(h->ev_gin);
    if (h->ev_gout) cudaEventDestroy(h->ev_gout);
    if (h->s1) cudaStreamDestroy(h->s1);
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    if (h->h_scal) cudaFreeHost(h->h_scal);
    if (h->h_sums) cudaFreeHost(h->h_sums);
    if (h->h_diag) cudaFreeHost(h->h_diag);
    if (h->h_status) cudaFreeHost(h->h_status);
    if (h->prof_ev) {
        for (cudaEvent_t e : *h->prof_ev) cudaEventDestroy(e);
        delete h->prof_ev;
        delete h->prof_slot;
    }
    delete h->xi;
    delete h->xi2;
    delete h->seed;
    delete h;
    return PIMD_OK;
}

int pimd_set_stream(pimd_t h, void *cuda_stream)
{
    if (!h) return PIMD_EINVAL;
    h->s0 = (cudaStream_t)cuda_stream;
    return PIMD_OK;
}

size_t pimd_workspace_bytes(pimd_t h)
{
    if (!h) return 0;
    pimd_s tmp = *h;
    return carve(&tmp, nullptr);
}

int pimd_set_workspace(pimd_t h, void *dev_ptr, size_t bytes)
{
    if (!h) return PIMD_EINVAL;
    if (h->carved) return fail(h, PIMD_EINVAL, "workspace already in use");
    if (!dev_ptr || ((uintptr_t)dev_ptr & 255)) return fail(h, PIMD_EINVAL, "workspace must be a 256-byte aligned device pointer");
    if (bytes < pimd_workspace_bytes(h)) return fail(h, PIMD_ENOMEM, "workspace too small: %zu < %zu", bytes, pimd_workspace_bytes(h));
    h->ws = (unsigned char *)dev_ptr;
    h->ws_bytes = bytes;
    h->own_ws = false;
    return PIMD_OK;
}

int pimd_set_gamma(pimd_t h, double gamma)
{
    if (!h) return PIMD_EINVAL;
    if (!(gamma > 0) || !std::isfinite(gamma)) return fail(h, PIMD_EINVAL, "gamma must be positive");
    if (gamma != h->gamma) drop_graphs(h); // the captured integrator nodes carry the friction as kernel arguments
    h->gamma = gamma;
    return PIMD_OK;
}

int pimd_set_concurrency(pimd_t h, int on)
{
    if (!h) return PIMD_EINVAL;
    h->concurrent = on != 0;
    return PIMD_OK;
}

int pimd_set_species(pimd_t h, int nspecies, const int *counts)
{
    if (!h) return PIMD_EINVAL;
    if (h->carved) return fail(h, PIMD_EINVAL, "pimd_set_species must precede the first state / compute call");
    if (nspecies < 1 || nspecies > PIMD_MAX_SPECIES || !counts) return fail(h, PIMD_EINVAL, "need 1 <= nspecies <= %d", PIMD_MAX_SPECIES);
    long long tot = 0;
    for (int k = 0; k < nspecies; ++k) {
        if (counts[k] < 1) return fail(h, PIMD_EINVAL, "every species needs at least one particle");
        tot += counts[k];
    }
    if (tot != h->N) return fail(h, PIMD_EINVAL, "species counts add up to %lld, not N = %d", tot, h->N);
    const int old_n = h->nspecies;
    int old_counts[PIMD_MAX_SPECIES];
    for (int k = 0; k < PIMD_MAX_SPECIES; ++k) old_counts[k] = h->counts[k];
    h->nspecies = nspecies;
    for (int k = 0; k < nspecies; ++k) h->counts[k] = counts[k];
    const int rc = setup_species(h);
    if (rc) { // the batch leaves no room for the panel workers these species need: keep the previous partition
        char msg[512];
        std::snprintf(msg, sizeof msg, "%s", h->err);
        h->nspecies = old_n;
        for (int k = 0; k < PIMD_MAX_SPECIES; ++k) h->counts[k] = old_counts[k];
        setup_species(h);
        std::snprintf(h->err, sizeof h->err, "%s", msg);
    }
    return rc;
}

int pimd_set_pair_potential(pimd_t h, int kind)
{
    if (!h) return PIMD_EINVAL;
    if (kind != PIMD_PAIR_GAUSSIAN && kind != PIMD_PAIR_SOFT_COULOMB) return fail(h, PIMD_EINVAL, "unknown pair potential %d", kind);
    if (kind != h->pot) { drop_graphs(h); h->forces_valid = false; }
    h->pot = kind;
    return PIMD_OK;
}

int pimd_set_pair_histogram(pimd_t h, int nbins, double rmax)
{
    if (!h) return PIMD_EINVAL;
    if (nbins < 0 || nbins > MAX_BINS || (nbins > 0 && !(rmax > 0))) return fail(h, PIMD_EINVAL, "need 0 <= nbins <= %d and rmax > 0", MAX_BINS);
    h->nbins_gr = nbins;
    h->rmax_gr = rmax;
    return PIMD_OK;
}

// copies between the caller's contiguous [B][n] doubles and the replica regions (rstride apart)
static int copy_in(pimd_t h, double *dst, const double *src, size_t n, cudaMemcpyKind kind)
{
    CU(cudaMemcpy2DAsync(dst, h->rstride, src, n * 8, n * 8, (size_t)h->B, kind, h->s0));
    return PIMD_OK;
}
static int copy_out(pimd_t h, double *dst, const double *src, size_t n, cudaMemcpyKind kind)
{
    CU(cudaMemcpy2DAsync(dst, n * 8, src, h->rstride, n * 8, (size_t)h->B, kind, h->s0));
    return PIMD_OK;
}

static int set_state_impl(pimd_t h, const double *x, const double *v, cudaMemcpyKind kind)
{
    if (!h) return PIMD_EINVAL;
    if (!x) return fail(h, PIMD_EINVAL, "x is NULL");
    int rc = ensure_ws(h);
    if (rc) return rc;
    rc = copy_in(h, h->x, x, h->ndof, kind);
    if (rc) return rc;
    if (v) rc = copy_in(h, h->v, v, h->ndof, kind);
    else CU(cudaMemset2DAsync(h->v, h->rstride, 0, h->ndof * 8, (size_t)h->B, h->s0));
    if (rc) return rc;
    if (h->thermostat == PIMD_THERMOSTAT_NHC) CU(cudaMemset2DAsync(h->nhc, h->rstride, 0, h->ndof * 8 * PIMD_NHC_LENGTH, (size_t)h->B, h->s0));
    CU(cudaMemset2DAsync(h->istatus, h->rstride, 0, 4, (size_t)h->B, h->s0));
    for (int set = 0; set < 2; ++set)
        for (int sp = 0; sp < h->nspecies; ++sp) CU(cudaMemset2DAsync(h->ex[set][sp].p.status, h->rstride, 0, 8, (size_t)h->B, h->s0));
    h->forces_valid = false;
    h->tables_valid = false;
    h->scalars_valid = false;
    h->shard_imported = false;
    for (int set = 0; set < 2; ++set)
        for (int sp = 0; sp < h->nspecies; ++sp) h->ex[set][sp].history = 0; // a new trajectory: no extrapolation
    // The exchange gauge of the last evaluation is kept: the stale-gauge kernel accepts it only if every row sum stays
    // within 2^+-64 of it (chain_cta_spec) and otherwise redoes the recursion with a fresh max-plus gauge.
    return PIMD_OK;
}

static int get_state_impl(pimd_t h, double *x, double *v, cudaMemcpyKind kind)
{
    if (!h) return PIMD_EINVAL;
    int rc = ensure_ws(h);
    if (rc) return rc;
    if (x && (rc = copy_out(h, x, h->x, h->ndof, kind))) return rc;
    if (v && (rc = copy_out(h, v, h->v, h->ndof, kind))) return rc;
    CU(cudaStreamSynchronize(h->s0));
    return PIMD_OK;
}

int pimd_set_state(pimd_t h, const double *x_dev, const double *v_dev) { return set_state_impl(h, x_dev, v_dev, cudaMemcpyDeviceToDevice); }
int pimd_get_state(pimd_t h, double *x_dev, double *v_dev) { return get_state_impl(h, x_dev, v_dev, cudaMemcpyDeviceToDevice); }
int pimd_set_state_host(pimd_t h, const double *x_host, const double *v_host) { return set_state_impl(h, x_host, v_host, cudaMemcpyHostToDevice); }
int pimd_get_state_host(pimd_t h, double *x_host, double *v_host) { return get_state_impl(h, x_host, v_host, cudaMemcpyDeviceToHost); }

int pimd_get_step_count(pimd_t h, uint64_t *step_host)
{
    if (!h || !step_host) return PIMD_EINVAL;
    *step_host = h->step;
    return PIMD_OK;
}
int pimd_set_step_count(pimd_t h, uint64_t step)
{
    if (!h) return PIMD_EINVAL;
    h->step = step;
    return PIMD_OK;
}
int pimd_get_nhc(pimd_t h, double *nhc_dev)
{
    if (!h || !nhc_dev) return PIMD_EINVAL;
    if (h->thermostat != PIMD_THERMOSTAT_NHC) return fail(h, PIMD_EINVAL, "thermostat is not Nose-Hoover");
    int rc = ensure_ws(h);
    if (rc) return rc;
    rc = copy_out(h, nhc_dev, h->nhc, h->ndof * PIMD_NHC_LENGTH, cudaMemcpyDeviceToDevice);
    if (rc) return rc;
    CU(cudaStreamSynchronize(h->s0));
    return PIMD_OK;
}
int pimd_set_nhc(pimd_t h, const double *nhc_dev)
{
    if (!h || !nhc_dev) return PIMD_EINVAL;
    if (h->thermostat != PIMD_THERMOSTAT_NHC) return fail(h, PIMD_EINVAL, "thermostat is not Nose-Hoover");
    int rc = ensure_ws(h);
    if (rc) return rc;
    return copy_in(h, h->nhc, nhc_dev, h->ndof * PIMD_NHC_LENGTH, cudaMemcpyDeviceToDevice);
}

static int launch_combine(pimd_t h, double *dst)
{
    const int own_first = (!h->sharded || h->j0 == 0) ? 1 : 0, own_last = (!h->sharded || h->j0 + h->P == h->Pg) ? 1 : 0;
    {
        ProfScope ps(h, PIMD_PROF_COMBINE, h->s0);
        k_combine<<<dim3((unsigned)((h->ndof + 255) / 256), h->B), 256, 0, h->s0>>>(dst, h->F, h->Fex1, h->FexP, h->ndof, h->slice, h->P,
                                                                                   own_first, own_last, h->rstride);
    }
    CU(cudaGetLastError());
    return PIMD_OK;
}

// V_B and sign per replica from the species' scalars: V = sum over species, sign = product
static int fetch_scalars(pimd_t h, double *vb, int *sign)
{
    const size_t B = (size_t)h->B;
    CU(cudaMemcpy2DAsync(h->h_scal, sizeof(Scalars) * PIMD_MAX_SPECIES, h->scal[0], h->rstride, sizeof(Scalars) * PIMD_MAX_SPECIES, B,
                         cudaMemcpyDeviceToHost, h->s0));
    int rc = read_status(h);
    if (rc) return rc;
    for (size_t b = 0; b < B; ++b) {
        double v = 0.0, sg = 1.0;
        for (int sp = 0; sp < h->nspecies; ++sp) {
            v += h->h_scal[b * PIMD_MAX_SPECIES + sp].vb;
            sg *= h->h_scal[b * PIMD_MAX_SPECIES + sp].sign;
        }
        if (!std::isfinite(v)) return fail(h, PIMD_ENUMERIC, "V_B is not finite");
        if (vb) vb[b] = v;
        if (sign) sign[b] = sg < 0 ? -1 : 1;
    }
    return PIMD_OK;
}

static int forces_impl(pimd_t h, double *f, bool host, double *vb, int *sign)
{
    if (!h) return PIMD_EINVAL;
    if (h->sharded) return fail(h, PIMD_EINVAL, "bead shard: use pimd_shard_forces");
    int rc = eval_forces(h, true, false, 0, 0.0);
    if (rc) return rc;
    if (f) {
        rc = launch_combine(h, host ? h->Fout : f);
        if (rc) return rc;
        if (host) CU(cudaMemcpyAsync(f, h->Fout, (size_t)h->B * h->ndof * 8, cudaMemcpyDeviceToHost, h->s0));
    }
    return fetch_scalars(h, vb, sign);
}

static int get_forces_impl(pimd_t h, double *f, bool host)
{
    if (!h || !f) return PIMD_EINVAL;
    if (!h->forces_valid) return fail(h, PIMD_EINVAL, "no forces cached for the current positions");
    int rc = launch_combine(h, host ? h->Fout : f);
    if (rc) return rc;
    if (host) CU(cudaMemcpyAsync(f, h->Fout, (size_t)h->B * h->ndof * 8, cudaMemcpyDeviceToHost, h->s0));
    CU(cudaStreamSynchronize(h->s0));
    return PIMD_OK;
}

static int set_forces_impl(pimd_t h, const double *f, cudaMemcpyKind kind)
{
    if (!h || !f) return PIMD_EINVAL;
    int rc = ensure_ws(h);
    if (rc) return rc;
    rc = copy_in(h, h->F, f, h->ndof, kind);
    if (rc) return rc;
    CU(cudaMemset2DAsync(h->Fex1, h->rstride, 0, h->slice * 8, (size_t)h->B, h->s0));
    CU(cudaMemset2DAsync(h->FexP, h->rstride, 0, h->slice * 8, (size_t)h->B, h->s0));
    h->forces_valid = true;
    return PIMD_OK;
}

int pimd_get_forces(pimd_t h, double *f_dev) { return get_forces_impl(h, f_dev, false); }
int pimd_get_forces_host(pimd_t h, double *f_host) { return get_forces_impl(h, f_host, true); }
int pimd_set_forces(pimd_t h, const double *f_dev) { return set_forces_impl(h, f_dev, cudaMemcpyDeviceToDevice); }
int pimd_set_forces_host(pimd_t h, const double *f_host) { return set_forces_impl(h, f_host, cudaMemcpyHostToDevice); }

int pimd_forces(pimd_t h, double *f_dev, double *vb, int *sign) { return forces_impl(h, f_dev, false, vb, sign); }
int pimd_forces_host(pimd_t h, double *f_host, double *vb, int *sign) { return forces_impl(h, f_host, true, vb, sign); }

int pimd_get_tables(pimd_t h, double *vfwd, double *vbwd, double *pnext)
{
    if (!h) return PIMD_EINVAL;
    if (h->B != 1 || h->nspecies != 1) return fail(h, PIMD_EINVAL, "tables are reported for one replica and one species");
    if (!h->tables_valid) return fail(h, PIMD_EINVAL, "no force evaluation to report");
    if ((vfwd || vbwd) && h->all_zero[0]) return fail(h, PIMD_EINVAL, "tables are not formed for xi = 0");
    const ExchPtrs &ex = h->ex[0][0].p;
    const int N = h->N;
    const double lambda = (*h->xi)[0] != 0.0 ? std::log(std::fabs((*h->xi)[0])) : 0.0;
    if (pnext) CU(cudaMemcpyAsync(pnext, ex.pnext, (size_t)N * 8, cudaMemcpyDeviceToHost, h->s0));
    if (vfwd || vbwd) {
        // V^{[1,n]} and V^{[u,N]} from the de-trended tables g: prefix sums of E_int and C(l,l+1)
        // are diagnostics of the evaluation, formed here in long double.
        std::vector<double> gf(2 * (size_t)(N + 1)), gb(2 * (size_t)(N + 1)), zf(N + 1), zb(N + 1), eint(N), cnext(N);
        double rf[4];
        CU(cudaMemcpyAsync(gf.data(), ex.g[0], (size_t)(N + 1) * 16, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(gb.data(), ex.g[1], (size_t)(N + 1) * 16, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(zf.data(), ex.gs[0], (size_t)(N + 1) * 8, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(zb.data(), ex.gs[1], (size_t)(N + 1) * 8, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(eint.data(), ex.eint, (size_t)N * 8, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(cnext.data(), ex.cnext, (size_t)N * 8, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(rf, ex.rfin, 32, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaStreamSynchronize(h->s0));
        const long double beta = h->beta, lam = lambda;
        std::vector<long double> S(N + 1), T(N + 1); // 1-based: S[0] = 0, T[v] = S[v-1] + E_int[v], S[v] = T[v] + C[v][v+1]
        S[0] = 0;
        for (int v = 1; v <= N; ++v) {
            T[v] = S[v - 1] + eint[v - 1];
            S[v] = T[v] + (v < N ? (long double)cnext[v - 1] / beta : 0.0L);
        }
        // g_j = T_j + log|Zhat_j| (the recursion carries the gauge T and the linear factor Zhat)
        auto gfv = [&](int j) -> long double { return j < N ? (long double)gf[2 * j] + gf[2 * j + 1] + logl(fabsl((long double)zf[j])) : 0.0L; };
        auto gbv = [&](int j) -> long double { return (long double)gb[2 * j] + gb[2 * j + 1] + logl(fabsl((long double)zb[j])); };
        if (vfwd) {
            vfwd[0] = 0.0;
            for (int n = 1; n <= N; ++n) {
                // a[n+1] = g^f_n = L_n + beta S[n] - (n+1) lambda ; for n = N use R_N
                long double L;
                if (n < N) L = gfv(n) - beta * S[n] + (long double)(n + 1) * lam;
                else L = ((long double)rf[0] + rf[1]) - beta * T[N] + (long double)N * lam - logl((long double)N);
                vfwd[n] = (double)(-L / beta);
            }
        }
        if (vbwd) {
            // qhat[l] = g^b_{N-l} (1-based l), q[l] = qhat[l] + q[N], q[N] = -beta T[N] + N lambda - ln N,
            // M_{l+1} = q[l] + beta T[l] - l lambda + ln l ;  M_1 = L_N
            const long double qN = -beta * T[N] + (long double)N * lam - logl((long double)N);
            vbwd[0] = 0.0;
            vbwd[N + 1] = 0.0;
            for (int l = 1; l <= N; ++l) {
                const long double M = gbv(N - l) + qN + beta * T[l] - (long double)l * lam + logl((long double)l);
                if (l + 1 <= N) vbwd[l + 1] = (double)(-M / beta);
            }
            const long double LN = ((long double)rf[0] + rf[1]) - beta * T[N] + (long double)N * lam - logl((long double)N);
            vbwd[1] = (double)(-LN / beta);
        }
    } else {
        CU(cudaStreamSynchronize(h->s0));
    }
    return PIMD_OK;
}

static int nxn_check(pimd_t h, const void *out)
{
    if (!h || !out) return PIMD_EINVAL;
    if (h->B != 1 || h->nspecies != 1 || h->sharded) return fail(h, PIMD_EINVAL, "N x N output: one replica, one species, no bead shards");
    if (h->N > 65535) return fail(h, PIMD_EINVAL, "N x N output supported up to N = 65535");
    return ensure_ws(h);
}

int pimd_cycle_energies(pimd_t h, double *e_dev)
{
    int rc = nxn_check(h, e_dev);
    if (rc) return rc;
    switch (h->d) {
    case 1: return cycle_energies_impl<1>(h, e_dev);
    case 2: return cycle_energies_impl<2>(h, e_dev);
    default: return cycle_energies_impl<3>(h, e_dev);
    }
}

int pimd_connection_probabilities(pimd_t h, double *pr_dev)
{
    int rc = nxn_check(h, pr_dev);
    if (rc) return rc;
    if (!h->tables_valid) {
        rc = eval_forces(h, false, false, 0, 0.0);
        if (rc) return rc;
    }
    switch (h->d) {
    case 1: rc = prmat_impl<1>(h, pr_dev); break;
    case 2: rc = prmat_impl<2>(h, pr_dev); break;
    default: rc = prmat_impl<3>(h, pr_dev); break;
    }
    if (rc) return rc;
    CU(cudaGetLastError());
    return read_status(h);
}

int pimd_step(pimd_t h, int nsteps)
{
    if (!h) return PIMD_EINVAL;
    if (nsteps < 0) return fail(h, PIMD_EINVAL, "nsteps < 0");
    return run_steps(h, nsteps, 0, 0, 0.0);
}

int pimd_run(pimd_t h, int nsteps, int est_every, int nbins, double rmax)
{
    if (!h) return PIMD_EINVAL;
    if (nsteps < 0 || est_every < 0) return fail(h, PIMD_EINVAL, "nsteps < 0 or est_every < 0");
    if (nbins < 0 || nbins > MAX_BINS || (nbins > 0 && !(rmax > 0))) return fail(h, PIMD_EINVAL, "nbins must be in [0, %d] with rmax > 0", MAX_BINS);
    return run_steps(h, nsteps, est_every, nbins, rmax);
}

int pimd_read_accumulators(pimd_t h, double *nsamples, double *sum_eprim, double *sum_evir, double *hist_sum, int nbins,
                           double *gr_sum, int nbins_gr, int reset)
{
    if (!h) return PIMD_EINVAL;
    if (nbins < 0 || nbins > MAX_BINS || nbins_gr < 0 || nbins_gr > MAX_BINS) return fail(h, PIMD_EINVAL, "bad bin count");
    int rc = ensure_ws(h);
    if (rc) return rc;
    const size_t B = (size_t)h->B;
    CU(cudaMemcpy2DAsync(h->h_sums, sizeof(EstSums), h->sums, h->rstride, sizeof(EstSums), B, cudaMemcpyDeviceToHost, h->s0));
    if (hist_sum && nbins > 0) CU(cudaMemcpy2DAsync(hist_sum, (size_t)nbins * 8, h->hist_acc, h->rstride, (size_t)nbins * 8, B, cudaMemcpyDeviceToHost, h->s0));
    if (gr_sum && nbins_gr > 0) CU(cudaMemcpy2DAsync(gr_sum, (size_t)nbins_gr * 8, h->gr_acc, h->rstride, (size_t)nbins_gr * 8, B, cudaMemcpyDeviceToHost, h->s0));
    if (reset) {
        CU(cudaMemset2DAsync(h->sums, h->rstride, 0, sizeof(EstSums), B, h->s0));
        CU(cudaMemset2DAsync(h->hist_acc, h->rstride, 0, (size_t)MAX_BINS * 8, B, h->s0));
        CU(cudaMemset2DAsync(h->gr_acc, h->rstride, 0, (size_t)MAX_BINS * 8, B, h->s0));
    }
    rc = read_status(h); // synchronises
    if (rc) return rc;
    for (size_t b = 0; b < B; ++b) {
        if (nsamples) nsamples[b] = h->h_sums[b].n;
        if (sum_eprim) sum_eprim[b] = h->h_sums[b].sum_ep;
        if (sum_evir) sum_evir[b] = h->h_sums[b].sum_ev;
    }
    return PIMD_OK;
}

int pimd_estimators(pimd_t h, double *e_prim, double *e_vir, double *hist, int nbins, double rmax)
{
    if (!h) return PIMD_EINVAL;
    if (nbins < 0 || nbins > MAX_BINS) return fail(h, PIMD_EINVAL, "nbins must be in [0, %d]", MAX_BINS);
    if (nbins > 0 && (!hist || !(rmax > 0))) return fail(h, PIMD_EINVAL, "hist is NULL or rmax <= 0");
    int rc = eval_forces(h, true, true, nbins, rmax);
    if (rc == PIMD_OK) rc = launch_estimate(h, nbins, false);
    if (rc) return rc;
    const size_t B = (size_t)h->B;
    CU(cudaMemcpy2DAsync(h->h_sums, sizeof(EstSums), h->sums, h->rstride, sizeof(EstSums), B, cudaMemcpyDeviceToHost, h->s0));
    if (nbins > 0) CU(cudaMemcpy2DAsync(hist, (size_t)nbins * 8, h->hist, h->rstride, (size_t)nbins * 8, B, cudaMemcpyDeviceToHost, h->s0));
    rc = read_status(h);
    if (rc) return rc;
    for (size_t b = 0; b < B; ++b) {
        if (e_prim) e_prim[b] = h->h_sums[b].last_ep;
        if (e_vir) e_vir[b] = h->h_sums[b].last_ev;
    }
    return PIMD_OK;
}

int pimd_pair_histogram(pimd_t h, double *gr_host)
{
    if (!h || !gr_host) return PIMD_EINVAL;
    if (h->nbins_gr <= 0) return fail(h, PIMD_EINVAL, "pimd_set_pair_histogram first");
    if (!h->carved) return fail(h, PIMD_EINVAL, "no estimator evaluation yet");
    CU(cudaMemcpy2DAsync(gr_host, (size_t)h->nbins_gr * 8, h->gr, h->rstride, (size_t)h->nbins_gr * 8, (size_t)h->B, cudaMemcpyDeviceToHost, h->s0));
    CU(cudaStreamSynchronize(h->s0));
    return PIMD_OK;
}

int pimd_reweight(pimd_t h, const double *xi_obs, double *ln_abs_r, int *sign, double *eps_obs, double *eps_samp)
{
    if (!h || !xi_obs) return PIMD_EINVAL;
    if (h->sharded) return fail(h, PIMD_EINVAL, "pimd_reweight is not available on a bead shard");
    int rc = ensure_ws(h);
    if (rc) return rc;
    bool any0 = false, anynz = false, same = true;
    for (int b = 0; b < h->B; ++b) {
        if (!std::isfinite(xi_obs[b])) return fail(h, PIMD_EINVAL, "xi_obs must be finite");
        if (xi_obs[b] == 0.0) any0 = true; else anynz = true;
        same = same && xi_obs[b] == (*h->xi2)[b];
    }
    if (any0 && anynz) return fail(h, PIMD_EINVAL, "xi_obs is either all 0 or all != 0");
    if (!same) {
        h->xi2->assign(xi_obs, xi_obs + h->B);
        rc = upload_params(h, 1);
        if (rc) return rc;
        for (int sp = 0; sp < h->nspecies; ++sp) h->ex[1][sp].gauge_valid = false;
    }
    // the sampling xi's tables and scalars at the current positions
    if (!h->tables_valid) {
        rc = eval_forces(h, true, false, 0, 0.0);
        if (rc) return rc;
    } else if (!h->scalars_valid) {
        for (int sp = 0; sp < h->nspecies; ++sp) {
            ExchCtx &c = h->ex[0][sp];
            ProfScope ps(h, PIMD_PROF_FINALIZE, h->s0);
            k_finalize<256><<<h->B, 256, 0, h->s0>>>(c.N, c.nprep, c.nasm, h->beta, c.rp, std::lgamma((double)c.N + 1.0), c.p, c.ecpart, c.scal, h->rstride);
        }
        CU(cudaGetLastError());
        h->scalars_valid = true;
    }
    // the same recursion with xi_obs (second set of exchange tables; its exterior forces go to a scratch buffer)
    for (int sp = 0; sp < h->nspecies; ++sp) {
        rc = prep_d(h, h->ex[1][sp], h->s0);
        if (rc == PIMD_OK) rc = exchange_d(h, h->ex[1][sp], 1, h->s0, true);
        if (rc) return rc;
    }
    const size_t B = (size_t)h->B, row = sizeof(Scalars) * PIMD_MAX_SPECIES;
    std::vector<Scalars> obs(B * PIMD_MAX_SPECIES);
    CU(cudaMemcpy2DAsync(obs.data(), row, h->scal[1], h->rstride, row, B, cudaMemcpyDeviceToHost, h->s0));
    CU(cudaMemcpy2DAsync(h->h_scal, row, h->scal[0], h->rstride, row, B, cudaMemcpyDeviceToHost, h->s0));
    for (int sp = 0; sp < h->nspecies; ++sp)
        CU(cudaMemcpy2DAsync(h->h_status + B * (1 + PIMD_MAX_SPECIES + sp), 4, h->ex[1][sp].p.status, h->rstride, 4, B, cudaMemcpyDeviceToHost, h->s0));
    rc = read_status(h);
    if (rc) return rc;
    for (size_t b = 0; b < B; ++b) {
        double vo = 0.0, vs = 0.0, so = 1.0, ss = 1.0, eo = 0.0, es = 0.0;
        int st = 0;
        for (int sp = 0; sp < h->nspecies; ++sp) {
            const Scalars &o = obs[b * PIMD_MAX_SPECIES + sp], &q = h->h_scal[b * PIMD_MAX_SPECIES + sp];
            vo += o.vb; so *= o.sign; eo += o.ec;
            vs += q.vb; ss *= q.sign; es += q.ec;
            st |= h->h_status[B * (1 + PIMD_MAX_SPECIES + sp) + b];
        }
        if (st & ST_NODE) return fail(h, PIMD_ENUMERIC, "W(xi_obs) summed to zero (a node)");
        if (!std::isfinite(vo) || !std::isfinite(vs)) return fail(h, PIMD_ENUMERIC, "V_B is not finite");
        if (ln_abs_r) ln_abs_r[b] = -h->beta * (vo - vs);
        if (sign) sign[b] = (so * ss < 0) ? -1 : 1;
        if (eps_obs) eps_obs[b] = -eo;
        if (eps_samp) eps_samp[b] = -es;
    }
    return PIMD_OK;
}

// ---- bead shards ------------------------------------------------------------------------------------
int pimd_shard_layout(pimd_t h, int *j0, int *p_local, size_t *pack_doubles)
{
    if (!h) return PIMD_EINVAL;
    if (j0) *j0 = h->j0;
    if (p_local) *p_local = h->P;
    if (pack_doubles) *pack_doubles = pack_doubles_of(h->N, h->d);
    return PIMD_OK;
}

int pimd_shard_export(pimd_t h, double *send_dev)
{
    if (!h || !send_dev) return PIMD_EINVAL;
    if (!h->sharded) return fail(h, PIMD_EINVAL, "not a bead shard (pimd_create_sharded)");
    int rc = ensure_ws(h);
    if (rc) return rc;
    const unsigned grid = (unsigned)((h->N + 127) / 128);
    ProfScope ps(h, PIMD_PROF_SHARD, h->s0);
    switch (h->d) {
    case 1: k_shard_pack<1><<<grid, 128, 0, h->s0>>>(h->x, h->N, h->P, h->ks, send_dev); break;
    case 2: k_shard_pack<2><<<grid, 128, 0, h->s0>>>(h->x, h->N, h->P, h->ks, send_dev); break;
    default: k_shard_pack<3><<<grid, 128, 0, h->s0>>>(h->x, h->N, h->P, h->ks, send_dev); break;
    }
    CU(cudaGetLastError());
    return PIMD_OK;
}

static int shard_import(pimd_t h, const double *gathered_dev)
{
    const size_t packn = pack_doubles_of(h->N, h->d);
    CU(cudaMemcpyAsync(h->gathered, gathered_dev, (size_t)h->world * packn * 8, cudaMemcpyDeviceToDevice, h->s0));
    const unsigned grid = (unsigned)((h->N + 127) / 128);
    {
        ProfScope ps(h, PIMD_PROF_SHARD, h->s0);
        switch (h->d) {
        case 1: k_shard_eint<1><<<grid, 128, 0, h->s0>>>(h->gathered, h->N, h->world, packn, h->ks, h->eint_tot); break;
        case 2: k_shard_eint<2><<<grid, 128, 0, h->s0>>>(h->gathered, h->N, h->world, packn, h->ks, h->eint_tot); break;
        default: k_shard_eint<3><<<grid, 128, 0, h->s0>>>(h->gathered, h->N, h->world, packn, h->ks, h->eint_tot); break;
        }
    }
    CU(cudaGetLastError());
    h->shard_imported = true;
    return PIMD_OK;
}

int pimd_shard_forces(pimd_t h, const double *gathered_dev)
{
    if (!h || !gathered_dev) return PIMD_EINVAL;
    if (!h->sharded) return fail(h, PIMD_EINVAL, "not a bead shard (pimd_create_sharded)");
    int rc = ensure_ws(h);
    if (rc == PIMD_OK) rc = shard_import(h, gathered_dev);
    if (rc == PIMD_OK) rc = eval_forces(h, true, false, 0, 0.0);
    return rc;
}

int pimd_shard_scalars(pimd_t h, double *vb, int *sign)
{
    if (!h) return PIMD_EINVAL;
    if (!h->scalars_valid) return fail(h, PIMD_EINVAL, "no evaluation with scalars to report");
    return fetch_scalars(h, vb, sign);
}

int pimd_shard_begin_step(pimd_t h, double *send_dev)
{
    if (!h || !send_dev) return PIMD_EINVAL;
    if (!h->sharded) return fail(h, PIMD_EINVAL, "not a bead shard (pimd_create_sharded)");
    if (!h->forces_valid) return fail(h, PIMD_EINVAL, "bead shard: evaluate the forces of the starting state first (pimd_shard_export + pimd_shard_forces)");
    int rc = launch_integrate(h, false, true, 0, h->step);
    if (rc) return rc;
    h->forces_valid = false;
    h->tables_valid = false;
    h->scalars_valid = false;
    return pimd_shard_export(h, send_dev);
}

int pimd_shard_end_step(pimd_t h, const double *gathered_dev)
{
    if (!h || !gathered_dev) return PIMD_EINVAL;
    if (!h->sharded) return fail(h, PIMD_EINVAL, "not a bead shard (pimd_create_sharded)");
    int rc = shard_import(h, gathered_dev);
    if (rc == PIMD_OK) rc = eval_forces(h, false, false, 0, 0.0);
    if (rc == PIMD_OK) rc = launch_integrate(h, true, false, h->step, 0);
    if (rc) return rc;
    h->shard_imported = true; // close does not move the positions
    h->step++;
    return PIMD_OK;
}

int pimd_get_diagnostics(pimd_t h, uint64_t *out)
{
    if (!h || !out) return PIMD_EINVAL;
    int rc = ensure_ws(h);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h->h_diag, h->fallbacks, 8, cudaMemcpyDeviceToHost, h->s0));
    const int B = h->B, S = h->nspecies;
    for (int sp = 0; sp < S; ++sp)
        CU(cudaMemcpy2DAsync(h->h_status + (size_t)B * (1 + sp), 4, h->ex[0][sp].p.status + 1, h->rstride, 4, (size_t)B, cudaMemcpyDeviceToHost, h->s0));
    CU(cudaStreamSynchronize(h->s0));
    int sticky = 0;
    for (int k = B; k < B * (1 + S); ++k) sticky |= h->h_status[k];
    out[0] = h->h_diag[0];
    out[1] = (uint64_t)sticky;
    out[2] = (uint64_t)h->ex[0][0].nworkers;
    out[3] = (uint64_t)h->rstride;
    return PIMD_OK;
}

uint64_t pimd_launch_count(pimd_t h) { return h ? h->launches : 0; }

int pimd_set_profiling(pimd_t h, int on)
{
    if (!h) return PIMD_EINVAL;
    if (on < 0 || on > PIMD_PROFILE_PHASES) return fail(h, PIMD_EINVAL, "pimd_set_profiling: mode must be 0, PIMD_PROFILE_EVENTS or PIMD_PROFILE_PHASES");
    h->profiling = on != 0;
    h->phase_clock = on == PIMD_PROFILE_PHASES;
    return PIMD_OK;
}

int pimd_get_profile(pimd_t h, double *ms_host, uint64_t *count_host)
{
    if (!h) return PIMD_EINVAL;
    CU(cudaStreamSynchronize(h->s0));
    CU(cudaStreamSynchronize(h->s1));
    for (size_t i = 0; i < h->prof_slot->size(); ++i) {
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, (*h->prof_ev)[2 * i], (*h->prof_ev)[2 * i + 1]));
        h->prof_ms[(*h->prof_slot)[i]] += ms;
        h->prof_n[(*h->prof_slot)[i]]++;
    }
    h->prof_slot->clear(); // the events stay in the pool
    for (int k = 0; k < PIMD_PROF_NSLOTS; ++k) {
        if (ms_host) ms_host[k] = h->prof_ms[k];
        if (count_host) count_host[k] = h->prof_n[k];
        h->prof_ms[k] = 0.0;
        h->prof_n[k] = 0;
    }
    return PIMD_OK;
}

int pimd_get_chain_phases(pimd_t h, uint64_t *cycles_host)
{
    if (!h || !cycles_host) return PIMD_EINVAL;
    int rc = ensure_ws(h);
    if (rc) return rc;
    CU(cudaMemcpyAsync(cycles_host, h->phase, 16 * 8, cudaMemcpyDeviceToHost, h->s0));
    CU(cudaMemsetAsync(h->phase, 0, 16 * 8, h->s0));
    CU(cudaStreamSynchronize(h->s0));
    return PIMD_OK;
}

int pimd_selftest_exp(void *cuda_stream, int which, const double *x_dev, double *y_dev, size_t n)
{
    pimd_t h = nullptr;
    if (which < 0 || which > 3 || !x_dev || !y_dev) return fail(nullptr, PIMD_EINVAL, "pimd_selftest_exp: bad argument");
    if (n == 0) return PIMD_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    k_exp_selftest<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(x_dev, y_dev, n, which);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(st));
    return PIMD_OK;
}

int pimd_probe_fp64_peak(void *cuda_stream, double *tflops)
{
    pimd_t h = nullptr;
    if (!tflops) return PIMD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms * 8, iters = 4096;
    double *out = nullptr;
    CU(cudaMalloc((void **)&out, (size_t)blocks * 256 * 8));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        CU(cudaEventRecord(e0, st));
        k_dfma_probe<<<blocks, 256, 0, st>>>(out, iters, 1.0000001, 1e-9);
        CU(cudaEventRecord(e1, st));
        CU(cudaEventSynchronize(e1));
        float ms = 0;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    const double fmas = (double)blocks * 256 * (double)iters * 64.0;
    *tflops = 2.0 * fmas / (best * 1e-3) / 1e12;
    return PIMD_OK;
}

} // extern "C"

// ==========================================================================================================================
// pimd_cycle_energies_noalloc: the cycle-energy matrix of Eq. 7-10 for callers that must not allocate (include/pimd.h).
//
// The handle path (pimd_cycle_energies) keeps four O(N) tables in the handle's workspace: E_int, beta C(l,l+1), and their
// prefix sums S, T.  Here the same four tables live in the file-scope device array below, which is part of the library
// image: the driver sets it aside on every GPU when the library's module is loaded there and releases it when the process
// ends.  No cudaMalloc / cudaFree / cudaMallocHost, no stream or event creation, no handle.
//
// `g_noalloc_scratch` as host code sees it is only a stand-in for the device array (its host address means nothing to a
// kernel), so the entry point asks the runtime for the real device address -- cudaGetSymbolAddress, once per device, with that
// device current -- and hands that pointer to the kernels.
//
// Every table entry a call reads (indices < N) is written earlier in the same call, so nothing needs clearing between calls
// even though the array keeps the previous call's contents.  All calls on one GPU share the array: two calls whose kernels
// can overlap on the GPU (different streams, or two host threads) overwrite each other's tables.
// ==========================================================================================================================
// E_int | beta C(l,l+1) | S | T, PIMD_NOALLOC_MAX_N doubles each: 4 x 16384 x 8 B = 512 KiB on every GPU that loads the library
static __device__ __align__(256) double g_noalloc_scratch[4 * (size_t)PIMD_NOALLOC_MAX_N];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
double *g_noalloc_ptr[NOALLOC_MAX_DEVICES]; // device address of g_noalloc_scratch on device i, or nullptr: not looked up yet

// Variant of k_prep (step 3) that keeps only what Eq. 7-10 need and writes it to the scratch tables: E_int of every ring
// (Eq. 9) and the closing spring to the next particle, beta C(l,l+1) = kk |r_l^P - r_{l+1}^1|^2 (0 for the
// last particle).  x is [P][N][D]; one thread per particle.
template <int D>
__global__ void __launch_bounds__(128) k_noalloc_eint(const double *__restrict__ x, int N, int P, double ks, double kk,
                                                      double *__restrict__ eint, double *__restrict__ cnext_beta)
{
    const int l = blockIdx.x * 128 + threadIdx.x;
    if (l >= N) return;
    const size_t sl = (size_t)N * D;
    Vec<D> prev = ldvec<D>(x, l);
    double acc = 0.0;
    for (int j = 1; j < P; ++j) {
        const Vec<D> cur = ldvec<D>(x + (size_t)j * sl, l);
        acc += dist2<D>(cur, prev);
        prev = cur;
    }
    eint[l] = 0.5 * ks * acc;
    cnext_beta[l] = (l < N - 1) ? kk * dist2<D>(prev, ldvec<D>(x, l + 1)) : 0.0; // prev = bead P of particle l
}

// device address of the scratch array on the current device (looked up on the first call per device)
int noalloc_scratch(double **out)
{
    pimd_t h = nullptr;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(nullptr, PIMD_EINVAL, "pimd_cycle_energies_noalloc: device ordinal %d not supported", dev);
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p) return fail(nullptr, PIMD_ECUDA, "pimd_cycle_energies_noalloc: cudaGetSymbolAddress returned a null address");
        g_noalloc_ptr[dev] = (double *)p;
    }
    *out = g_noalloc_ptr[dev];
    return PIMD_OK;
}

template <int D> int cycle_energies_noalloc_impl(cudaStream_t st, const double *x_dev, int N, int P, double beta, double *scratch, double *e_dev)
{
    pimd_t h = nullptr;
    const double ks = (double)P / (beta * beta), kk = (double)P / (2.0 * beta); // as in create_impl
    double *eint = scratch, *cnb = scratch + PIMD_NOALLOC_MAX_N, *S = scratch + 2 * (size_t)PIMD_NOALLOC_MAX_N,
           *T = scratch + 3 * (size_t)PIMD_NOALLOC_MAX_N;
    k_noalloc_eint<D><<<(N + 127) / 128, 128, 0, st>>>(x_dev, N, P, ks, kk, eint, cnb);
    CU(cudaGetLastError());
    k_prefix_st<<<1, 1024, 0, st>>>(N, beta, eint, cnb, S, T);
    CU(cudaGetLastError());
    // bead P / bead 1 slices straight from the caller's x (the handle path reads its own copies rho[0] / sig[0])
    k_emat<D><<<dim3((N + 1023) / 1024, N), 256, 0, st>>>(N, ks, x_dev + (size_t)(P - 1) * N * D, x_dev, S, T, e_dev);
    CU(cudaGetLastError());
    return PIMD_OK;
}

} // namespace

extern "C" int pimd_cycle_energies_noalloc(void *cuda_stream, const double *x_dev, int N, int P, int d, double beta, double *e_dev)
{
    if (!x_dev || !e_dev) return fail(nullptr, PIMD_EINVAL, "pimd_cycle_energies_noalloc: x_dev and e_dev must not be NULL");
    if (N < 1 || P < 2 || d < 1 || d > 3 || !std::isfinite(beta) || !(beta > 0))
        return fail(nullptr, PIMD_EINVAL, "pimd_cycle_energies_noalloc: need N >= 1, P >= 2, d in {1,2,3}, beta > 0 (got N=%d P=%d d=%d beta=%g)", N, P, d, beta);
    if (N > PIMD_NOALLOC_MAX_N)
        return fail(nullptr, PIMD_EINVAL,
                    "pimd_cycle_energies_noalloc: N = %d exceeds PIMD_NOALLOC_MAX_N = %d, the size of the built-in scratch tables; "
                    "use pimd_cycle_energies (handle with a workspace) for larger systems", N, PIMD_NOALLOC_MAX_N);
    if ((((size_t)x_dev) & 15) != 0 || (((size_t)e_dev) & 7) != 0)
        return fail(nullptr, PIMD_EINVAL, "pimd_cycle_energies_noalloc: x_dev must be 16-byte aligned, e_dev 8-byte aligned");
    double *scratch = nullptr;
    int rc = noalloc_scratch(&scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    switch (d) {
    case 1: return cycle_energies_noalloc_impl<1>(st, x_dev, N, P, beta, scratch, e_dev);
    case 2: return cycle_energies_noalloc_impl<2>(st, x_dev, N, P, beta, scratch, e_dev);
    default: return cycle_energies_noalloc_impl<3>(st, x_dev, N, P, beta, scratch, e_dev);
    }
}
