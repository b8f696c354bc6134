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
#include <new>
#include <vector>

using namespace pimd;

namespace {

thread_local char g_create_error[512] = "";

constexpr int BEAD_TB = 128;
constexpr int PREP_TB = 64;
constexpr int ASM_TB = 128;
constexpr int MAX_BINS = 1 << 16;

} // namespace

struct pimd_s {
    int N, P, d;
    double beta, omega, g, s, xi, dt, gamma;
    int thermostat;
    uint64_t seed, step;
    // derived
    double ks, kk, lambda;
    size_t ndof, slice;
    int NB, nprep, nasm, look, look_spec, nworkers, sms;
    // streams
    cudaStream_t s0, s1;
    cudaEvent_t ev_fork, ev_join;
    bool concurrent;
    // memory
    unsigned char *ws;
    size_t ws_bytes;
    bool own_ws, carved;
    double *x, *v, *F, *Fout, *nhc, *Fex1, *FexP, *ecpart, *hist, *Sarr, *Tarr;
    ExchPtrs ex;
    Scalars *scal;
    EstAccum *est;
    int *status;
    unsigned long long *phase; // chain phase clock (profiling)
    unsigned long long *dstep; // MD step counter on the device (graph replay)
    // one MD step (force evaluation, then close + open) captured as a CUDA graph on an internal stream
    cudaStream_t sg;
    cudaEvent_t ev_gin, ev_gout;
    cudaGraphExec_t gexec;
    bool use_graph, graph_failed, graph_conc;
    uint64_t graph_launches;
    // pinned host mirrors
    Scalars *h_scal;
    EstAccum *h_est;
    int *h_status;
    bool forces_valid;
    bool tables_valid; // the exchange tables (g, gs, pnext, rfin) belong to the current positions
    bool gauge_valid; // g/gs hold the (T, Zhat) of a completed evaluation of nearby positions
    bool use_spec;    // PIMD_NOSPEC=1 turns the stale-gauge kernel off
    size_t spec_smem;
    int coop_max_blocks; // co-resident CTA limit of k_chain
    size_t chain_smem;
    uint64_t launches;
    // per-kernel device timing (pimd_set_profiling)
    bool profiling;
    std::vector<cudaEvent_t> *prof_ev;   // pairs (start, stop)
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

// carve the workspace; with base == nullptr only the size is computed
size_t carve(pimd_t h, unsigned char *base)
{
    size_t off = 0;
    auto take = [&](size_t bytes) -> unsigned char * {
        unsigned char *p = base ? base + off : nullptr;
        off = align_up(off + bytes, 256);
        return p;
    };
    const size_t N = (size_t)h->N, D = (size_t)h->d, nd = h->ndof;
    h->x = (double *)take(nd * 8);
    h->v = (double *)take(nd * 8);
    h->F = (double *)take(nd * 8);
    h->Fout = (double *)take(nd * 8);
    h->nhc = (double *)take(h->thermostat == PIMD_THERMOSTAT_NHC ? nd * 8 * PIMD_NHC_LENGTH : 8);
    h->Fex1 = (double *)take(N * D * 8);
    h->FexP = (double *)take(N * D * 8);
    for (int dir = 0; dir < 2; ++dir) {
        h->ex.rho[dir] = (double *)take(N * D * 8);
        h->ex.sig[dir] = (double *)take(N * D * 8);
        h->ex.cc[dir] = (double *)take(N * 8);
        h->ex.g[dir] = (double2 *)take((N + 1) * 16);
        h->ex.gs[dir] = (double *)take((N + 1) * 8);
        h->ex.pan_m[dir] = (double *)take(N * 8);
        h->ex.pan_s[dir] = (double *)take(N * 8);
        h->ex.panel_ready[dir] = (int *)take((size_t)h->NB * 4);
        h->ex.acc[dir] = (double *)take(N * (D + 2) * 8);
    }
    h->ex.cols_ready = (int *)take(2 * 4);
    h->ex.eint = (double *)take(N * 8);
    h->ex.cnext = (double *)take(N * 8);
    h->ex.cself = (double *)take(N * 8);
    h->ex.pnext = (double *)take(N * 8);
    h->ex.tpart = (double *)take((size_t)h->nprep * 2 * 8);
    h->ex.rfin = (double2 *)take(2 * 16);
    h->ex.rsgn = (double *)take(2 * 8);
    h->Sarr = (double *)take(N * 8);
    h->Tarr = (double *)take(N * 8);
    h->phase = (unsigned long long *)take(16 * 8);
    h->dstep = (unsigned long long *)take(8);
    h->status = (int *)take(4 * 4);
    h->ex.status = h->status;
    h->ecpart = (double *)take((size_t)h->nasm * 8);
    h->scal = (Scalars *)take(sizeof(Scalars));
    h->est = (EstAccum *)take(sizeof(EstAccum));
    h->hist = (double *)take((size_t)MAX_BINS * 8);
    return off;
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
    if (h->coop_max_blocks < 2) return fail(h, PIMD_ECUDA, "k_chain cannot be made co-resident (%d blocks)", h->coop_max_blocks);
    return PIMD_OK;
}

template <int D> int launch_bead(pimd_t h, cudaStream_t st, bool est, int nbins, double rmax)
{
    const dim3 grid((h->N + BEAD_TB - 1) / BEAD_TB, h->P), block(BEAD_TB);
    const double om2P = h->omega * h->omega / h->P, is2 = 1.0 / (h->s * h->s);
    {
        // spring + trap forces (and the trap energy / histogram on estimator calls): F is written here
        ProfScope ps(h, PIMD_PROF_BEAD, st);
        if (est) k_bead<D, false, true, BEAD_TB><<<grid, block, 0, st>>>(h->x, h->F, h->N, h->P, h->ks, om2P, is2, 0.0, h->g, h->est, h->hist, nbins, rmax);
        else k_bead<D, false, false, BEAD_TB><<<grid, block, 0, st>>>(h->x, h->F, h->N, h->P, h->ks, om2P, is2, 0.0, h->g, h->est, h->hist, nbins, rmax);
    }
    CU(cudaGetLastError());
    if (h->g != 0.0) {
        // pair forces, added to F (Newton's third law, one Gaussian per unordered pair)
        const int NT = (h->N + 31) / 32;
        const int hmax = (NT & 1) ? (NT - 1) / 2 : NT / 2;
        // offsets per task: small tasks balance small grids (measured: 1 is best up to N = 2500, 4 at N = 10000; tuning knob PIMD_PAIR_CH)
        int target = NT <= 100 ? 1 : (NT <= 200 ? 2 : 4);
        if (const char *e = std::getenv("PIMD_PAIR_CH")) { const int v = std::atoi(e); if (v >= 1 && v <= 64) target = v; }
        const int nchunk = hmax > 0 ? std::max(1, (hmax + target / 2) / target) : 0;
        const int ch = nchunk > 0 ? (hmax + nchunk - 1) / nchunk : 1;
        const long long tasks = (long long)NT * (nchunk + 1);
        const dim3 pgrid((unsigned)((tasks + PAIR_WARPS - 1) / PAIR_WARPS), h->P);
        const double coef = 2.0 * h->g / (h->s * h->P);
        ProfScope ps(h, PIMD_PROF_PAIR, st);
        if (est) k_pair<D, true><<<pgrid, PAIR_WARPS * 32, 0, st>>>(h->x, h->F, h->N, NT, nchunk, ch, 1.0 / h->s, coef, h->g, h->est);
        else k_pair<D, false><<<pgrid, PAIR_WARPS * 32, 0, st>>>(h->x, h->F, h->N, NT, nchunk, ch, 1.0 / h->s, coef, h->g, h->est);
    }
    CU(cudaGetLastError());
    return PIMD_OK;
}

template <int D> int launch_prep(pimd_t h, cudaStream_t st)
{
    {
        ProfScope ps(h, PIMD_PROF_PREP, st);
        k_prep<D, PREP_TB><<<h->nprep, PREP_TB * PREP_SPLIT, 0, st>>>(h->x, h->N, h->P, h->NB, h->ks, h->kk, h->lambda, h->ex);
    }
    CU(cudaGetLastError());
    return PIMD_OK;
}

template <int D> int launch_exchange(pimd_t h, cudaStream_t st, bool scalars)
{
    const bool sgn = h->xi < 0.0;
    if (h->xi == 0.0) {
        {
            ProfScope ps(h, PIMD_PROF_ASSEMBLE, st);
            k_exch_xi0<D, ASM_TB><<<h->nasm, ASM_TB, 0, st>>>(h->N, h->ks, h->ex, h->Fex1, h->FexP, h->ecpart);
        }
        CU(cudaGetLastError());
    } else {
        ChainArgs a;
        a.N = h->N; a.NB = h->NB; a.look = h->look; a.nworkers = h->nworkers;
        a.kk = h->kk; a.sx = sgn ? -1.0 : 1.0; a.p = h->ex;
        a.phase = h->profiling ? h->phase : nullptr;
        a.look_fb = h->look;
        const int look_spec = h->look_spec;
        void *args[] = {&a};
        const dim3 grid(1 + h->nworkers, 2), block(CH_THREADS);
        const void *fn = sgn ? (const void *)k_chain<D, true> : (const void *)k_chain<D, false>;
        if (h->gauge_valid && h->use_spec) {
            // the previous evaluation's gauge is at hand: linear pass only; the kernel redoes the recursion with a
            // fresh max-plus gauge itself (after a grid barrier) if the gauge turned out not to fit
            const void *fs = sgn ? (const void *)k_chain_spec<D, true> : (const void *)k_chain_spec<D, false>;
            a.look = look_spec; // the workers need one more block of head start when the chain runs this fast
            ProfScope ps(h, PIMD_PROF_CHAIN, st);
            CU(cudaLaunchCooperativeKernel(fs, grid, block, args, h->spec_smem, st));
        } else {
            ProfScope ps(h, PIMD_PROF_CHAIN, st);
            CU(cudaLaunchCooperativeKernel(fn, grid, block, args, h->chain_smem, st));
        }
        h->gauge_valid = true;
        const int NT = (h->N + FP_TB - 1) / FP_TB;
        // NT (NT+1) tiles at or below the diagonal (both directions); with fewer than 8 per SM one thread per row leaves
        // the kernel latency bound, so four threads share a row (measured at cfg3: 0.023 -> 0.017 ms with the columns cut
        // into four CTAs, less again with the partial sums combined inside one CTA)
        const long long tiles = (long long)NT * (NT + 1);
        const bool wide = tiles < 8LL * h->sms;
        const dim3 fgrid(wide ? (h->N + FP_TB / 4 - 1) / (FP_TB / 4) : NT, NT, 2);
        {
            ProfScope ps(h, PIMD_PROF_FORCEPASS, st);
            if (wide) {
                if (sgn) k_forcepass<D, true, 4><<<fgrid, FP_TB, 0, st>>>(h->N, h->kk, h->ex);
                else k_forcepass<D, false, 4><<<fgrid, FP_TB, 0, st>>>(h->N, h->kk, h->ex);
            } else {
                if (sgn) k_forcepass<D, true, 1><<<fgrid, FP_TB, 0, st>>>(h->N, h->kk, h->ex);
                else k_forcepass<D, false, 1><<<fgrid, FP_TB, 0, st>>>(h->N, h->kk, h->ex);
            }
        }
        CU(cudaGetLastError());
        {
            ProfScope ps(h, PIMD_PROF_ASSEMBLE, st);
            if (sgn) k_assemble<D, true, ASM_TB><<<h->nasm, ASM_TB, 0, st>>>(h->N, h->ks, h->xi, h->ex, h->Fex1, h->FexP, h->ecpart);
            else k_assemble<D, false, ASM_TB><<<h->nasm, ASM_TB, 0, st>>>(h->N, h->ks, h->xi, h->ex, h->Fex1, h->FexP, h->ecpart);
        }
        CU(cudaGetLastError());
    }
    if (scalars) {
        {
            ProfScope ps(h, PIMD_PROF_FINALIZE, st);
            k_finalize<256><<<1, 256, 0, st>>>(h->N, h->nprep, h->nasm, h->beta, h->lambda, h->xi, std::lgamma((double)h->N + 1.0),
                                               h->ex, h->ecpart, h->scal);
        }
        CU(cudaGetLastError());
    }
    return PIMD_OK;
}

// one force evaluation.  The exchange part stays on the main stream (k_prep, then the latency-bound
// k_chain, which must get its SMs first), the bead part (spring/trap/pair) is forked onto the helper
// stream after k_prep and fills the remaining SMs; joined before returning (in stream order).
int eval_forces(pimd_t h, bool scalars, bool est, int nbins, double rmax)
{
    int rc = ensure_ws(h);
    if (rc) return rc;
    if (est) {
        CU(cudaMemsetAsync(h->est, 0, sizeof(EstAccum), h->s0));
        if (nbins > 0) CU(cudaMemsetAsync(h->hist, 0, (size_t)nbins * 8, h->s0));
    }
    cudaStream_t sb = h->concurrent ? h->s1 : h->s0;
    switch (h->d) {
    case 1: rc = launch_prep<1>(h, h->s0); break;
    case 2: rc = launch_prep<2>(h, h->s0); break;
    default: rc = launch_prep<3>(h, h->s0); break;
    }
    if (rc) return rc;
    if (h->concurrent) {
        CU(cudaEventRecord(h->ev_fork, h->s0));
        CU(cudaStreamWaitEvent(h->s1, h->ev_fork, 0));
    }
    switch (h->d) {
    case 1: rc = launch_exchange<1>(h, h->s0, scalars); break;
    case 2: rc = launch_exchange<2>(h, h->s0, scalars); break;
    default: rc = launch_exchange<3>(h, h->s0, scalars); break;
    }
    if (rc) return rc;
    switch (h->d) {
    case 1: rc = launch_bead<1>(h, sb, est, nbins, rmax); break;
    case 2: rc = launch_bead<2>(h, sb, est, nbins, rmax); break;
    default: rc = launch_bead<3>(h, sb, est, nbins, rmax); break;
    }
    if (rc) return rc;
    if (h->concurrent) {
        CU(cudaEventRecord(h->ev_join, h->s1));
        CU(cudaStreamWaitEvent(h->s0, h->ev_join, 0));
    }
    h->forces_valid = true;
    h->tables_valid = true;
    return PIMD_OK;
}

int launch_integrate(pimd_t h, bool do_close, bool do_open, uint64_t step_close, uint64_t step_open, bool device_counter = false)
{
    const unsigned long long *dstep = device_counter ? h->dstep : nullptr;
    const double c1 = std::exp(-h->gamma * h->dt * 0.5);
    const double c2 = std::sqrt((1.0 - c1 * c1) / h->beta);
    const double Q = h->beta / (double)h->P;
    const unsigned grid = (unsigned)((h->ndof + 255) / 256);
#define LI(T) \
    k_integrate<T><<<grid, 256, 0, h->s0>>>(h->x, h->v, h->F, h->Fex1, h->FexP, h->nhc, h->ndof, h->slice, h->P, h->dt, c1, c2, \
                                            h->beta, Q, h->seed, step_close, step_open, do_close ? 1 : 0, do_open ? 1 : 0, h->status, dstep)
    {
        ProfScope ps(h, PIMD_PROF_INTEGRATE, h->s0);
        if (h->thermostat == PIMD_THERMOSTAT_LANGEVIN) LI(1);
        else if (h->thermostat == PIMD_THERMOSTAT_NHC) LI(2);
        else LI(0);
    }
#undef LI
    CU(cudaGetLastError());
    return PIMD_OK;
}

int read_status(pimd_t h)
{
    CU(cudaMemcpyAsync(h->h_status, h->status, 4 * sizeof(int), cudaMemcpyDeviceToHost, h->s0));
    CU(cudaStreamSynchronize(h->s0));
    const int st = h->h_status[0] | h->h_status[1];
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

} // namespace

// Capture "force evaluation ; close step s + open step s+1 ; counter += 1" once, on an internal stream (the caller's
// stream may be the legacy default stream, which cannot be captured).  Any failure (e.g. a driver that cannot put a
// cooperative launch into a graph) switches the feature off for this handle; nothing else depends on it.
static int ensure_graph(pimd_t h)
{
    if (h->gexec && h->graph_conc == h->concurrent) return PIMD_OK;
    if (h->graph_failed) return PIMD_ECUDA;
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    cudaStream_t user = h->s0;
    const uint64_t l0 = h->launches;
    const bool fv = h->forces_valid, tv = h->tables_valid;
    cudaGraph_t graph = nullptr;
    int rc = PIMD_OK;
    if (cudaStreamBeginCapture(h->sg, cudaStreamCaptureModeRelaxed) != cudaSuccess) rc = PIMD_ECUDA;
    if (rc == PIMD_OK) {
        h->s0 = h->sg;
        rc = eval_forces(h, false, false, 0, 0.0);
        if (rc == PIMD_OK) rc = launch_integrate(h, true, true, 0, 0, true);
        if (rc == PIMD_OK) {
            k_step_counter<<<1, 32, 0, h->sg>>>(h->dstep, 0ull, 1);
            h->launches++;
            if (cudaGetLastError() != cudaSuccess) rc = PIMD_ECUDA;
        }
        h->s0 = user;
        if (cudaStreamEndCapture(h->sg, &graph) != cudaSuccess || !graph) rc = PIMD_ECUDA;
    }
    if (rc == PIMD_OK && cudaGraphInstantiate(&h->gexec, graph, 0) != cudaSuccess) rc = PIMD_ECUDA;
    if (graph) cudaGraphDestroy(graph);
    h->graph_launches = h->launches - l0;
    h->launches = l0;
    h->forces_valid = fv;
    h->tables_valid = tv;
    if (rc != PIMD_OK) {
        cudaGetLastError();
        h->gexec = nullptr;
        h->graph_failed = true;
        return PIMD_ECUDA;
    }
    h->graph_conc = h->concurrent;
    return PIMD_OK;
}

template <int D> static int cycle_energies_impl(pimd_t h, double *e_dev)
{
    int rc = launch_prep<D>(h, h->s0); // E_int, C(l,l+1), bead-1 / bead-P slices of the current positions
    if (rc) return rc;
    k_prefix_st<<<1, 1024, 0, h->s0>>>(h->N, h->beta, h->ex.eint, h->ex.cnext, h->Sarr, h->Tarr);
    CU(cudaGetLastError());
    const dim3 grid((h->N + 1023) / 1024, h->N);
    {
        ProfScope ps(h, PIMD_PROF_EMAT, h->s0);
        k_emat<D><<<grid, 256, 0, h->s0>>>(h->N, h->ks, h->ex.rho[0], h->ex.sig[0], h->Sarr, h->Tarr, e_dev);
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(h->s0));
    return PIMD_OK;
}

template <int D> static int prmat_impl(pimd_t h, double *pr_dev)
{
    const dim3 grid((h->N + 1023) / 1024, h->N), gridp((h->N + 256 * PRMAT_COLS - 1) / (256 * PRMAT_COLS), (h->N + PRMAT_ROWS - 1) / PRMAT_ROWS);
    ProfScope ps(h, PIMD_PROF_PRMAT, h->s0);
    if (h->xi == 0.0) k_identity<<<grid, 256, 0, h->s0>>>(h->N, pr_dev);
    else if (h->xi < 0.0) k_prmat<D, true><<<gridp, 256, 0, h->s0>>>(h->N, h->kk, h->ex, pr_dev);
    else k_prmat<D, false><<<gridp, 256, 0, h->s0>>>(h->N, h->kk, h->ex, pr_dev);
    return PIMD_OK;
}

extern "C" {

const char *pimd_version(void) { return "pimd-b200 0.1 (sm_100a)"; }

const char *pimd_last_error(pimd_t h) { return h ? h->err : g_create_error; }

int pimd_create(pimd_t *out, int N, int P, int d, double beta, double omega, double g, double s, double xi, double dt,
                int thermostat, uint64_t seed)
{
    pimd_t h = nullptr;
    if (!out) return fail(nullptr, PIMD_EINVAL, "out is NULL");
    *out = nullptr;
    if (N < 1 || P < 2 || d < 1 || d > 3) return fail(nullptr, PIMD_EINVAL, "need N >= 1, P >= 2, d in {1,2,3} (got N=%d P=%d d=%d)", N, P, d);
    if (!finite_all({beta, omega, g, s, xi, dt}) || !(beta > 0) || !(s > 0) || !(dt > 0) || omega < 0)
        return fail(nullptr, PIMD_EINVAL, "need finite arguments with beta > 0, s > 0, dt > 0, omega >= 0");
    if (thermostat < 0 || thermostat > 2) return fail(nullptr, PIMD_EINVAL, "thermostat must be 0, 1 or 2");
    if ((double)N * P * d > 2.0e9) return fail(nullptr, PIMD_EINVAL, "N*P*d too large");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1)
        return fail(nullptr, PIMD_ECUDA, "no CUDA device (%s); libpimd has no CPU fallback", e != cudaSuccess ? cudaGetErrorString(e) : "count 0");
    h = new (std::nothrow) pimd_s();
    if (!h) return fail(nullptr, PIMD_ENOMEM, "host allocation failed");
    std::memset(h, 0, sizeof(*h));
    h->N = N; h->P = P; h->d = d;
    h->beta = beta; h->omega = omega; h->g = g; h->s = s; h->xi = xi; h->dt = dt; h->gamma = 1.0;
    h->thermostat = thermostat; h->seed = seed; h->step = 0;
    h->ks = (double)P / (beta * beta);          // m omega_P^2, omega_P = sqrt(P)/(beta hbar)
    h->kk = (double)P / (2.0 * beta);           // beta k_s / 2
    h->lambda = (xi != 0.0) ? std::log(std::fabs(xi)) : 0.0;
    h->slice = (size_t)N * d;
    h->ndof = h->slice * P;
    h->NB = (N + 31) / 32;
    h->nprep = (N + PREP_TB - 1) / PREP_TB;
    h->nasm = (N + ASM_TB - 1) / ASM_TB;
    h->look = 2;
    h->look_spec = 3;
    if (const char *e = std::getenv("PIMD_LOOK")) { // tuning knob: column blocks kept inside the chain CTA
        const int v = std::atoi(e);
        if (v >= 1 && v <= CH_MAXLOOK) h->look = h->look_spec = v;
    }
    h->concurrent = true;
    h->use_graph = !(std::getenv("PIMD_GRAPH") && std::atoi(std::getenv("PIMD_GRAPH")) == 0);
    h->gauge_valid = false;
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
    {
        // Panel workers per direction.  A worker spins while it waits for columns and owns a whole SM,
        // so only as many as the panel work needs are launched.
        const int want = h->NB - h->look - 1;
        int cap = h->coop_max_blocks / 2 - 1;
        // A worker needs about 480 NB cycles for its last row blocks and gets nworkers x (one chain block, about 3000
        // cycles) for each, so NB/5 workers keep the panels ahead of the chain; when the pair kernel dominates the step
        // (g != 0 and P N large: its work over the chain's grows like P N) the SMs are worth more there and NB/8 is enough.
        int need = (h->g != 0.0 && (long long)h->P * h->N > 80000) ? (h->NB + 7) / 8 : (h->NB + 4) / 5;
        if (const char *e = std::getenv("PIMD_WORKERS")) {
            const int v = std::atoi(e);
            if (v >= 1) need = v;
        }
        if (need > cap) need = cap;
        h->nworkers = want <= 0 ? 0 : (want < need ? want : need);
        if (want > 0 && h->nworkers < 1) return bail(fail(h, PIMD_ECUDA, "not enough co-resident CTAs for the recursion"));
    }
    if (cudaStreamCreateWithFlags(&h->s1, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&h->sg, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_gin, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_gout, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_scal, sizeof(Scalars)) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_est, sizeof(EstAccum)) != cudaSuccess ||
        cudaMallocHost((void **)&h->h_status, 4 * sizeof(int)) != cudaSuccess)
        return bail(fail(h, PIMD_ECUDA, "stream/event/pinned allocation failed: %s", cudaGetErrorString(cudaGetLastError())));
    *out = h;
    return PIMD_OK;
}

int pimd_destroy(pimd_t h)
{
    if (!h) return PIMD_OK;
    if (h->s0 || h->s1) cudaDeviceSynchronize();
    if (h->own_ws && h->ws) cudaFree(h->ws);
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    if (h->sg) cudaStreamDestroy(h->sg);
    if (h->ev_gin) cudaEventDestroy(h->ev_gin);
    if (h->ev_gout) cudaEventDestroy(h->ev_gout);
    if (h->s1) cudaStreamDestroy(h->s1);
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    if (h->h_scal) cudaFreeHost(h->h_scal);
    if (h->h_est) cudaFreeHost(h->h_est);
    if (h->h_status) cudaFreeHost(h->h_status);
    if (h->prof_ev) {
        for (cudaEvent_t e : *h->prof_ev) cudaEventDestroy(e);
        delete h->prof_ev;
        delete h->prof_slot;
    }
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
    h->gamma = gamma;
    return PIMD_OK;
}

int pimd_set_concurrency(pimd_t h, int on)
{
    if (!h) return PIMD_EINVAL;
    h->concurrent = on != 0;
    return PIMD_OK;
}

static int set_state_impl(pimd_t h, const double *x, const double *v, cudaMemcpyKind kind)
{
    if (!h) return PIMD_EINVAL;
    if (!x) return fail(h, PIMD_EINVAL, "x is NULL");
    int rc = ensure_ws(h);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h->x, x, h->ndof * 8, kind, h->s0));
    if (v) CU(cudaMemcpyAsync(h->v, v, h->ndof * 8, kind, h->s0));
    else CU(cudaMemsetAsync(h->v, 0, h->ndof * 8, h->s0));
    if (h->thermostat == PIMD_THERMOSTAT_NHC) CU(cudaMemsetAsync(h->nhc, 0, h->ndof * 8 * PIMD_NHC_LENGTH, h->s0));
    CU(cudaMemsetAsync(h->status, 0, 4 * sizeof(int), h->s0));
    h->forces_valid = false;
    h->tables_valid = false;
    // the exchange gauge of the last evaluation is kept: if the new positions are far from the old ones the
    // stale-gauge kernel notices and redoes the recursion with a fresh max-plus gauge
    return PIMD_OK;
}

static int get_state_impl(pimd_t h, double *x, double *v, cudaMemcpyKind kind)
{
    if (!h) return PIMD_EINVAL;
    int rc = ensure_ws(h);
    if (rc) return rc;
    if (x) CU(cudaMemcpyAsync(x, h->x, h->ndof * 8, kind, h->s0));
    if (v) CU(cudaMemcpyAsync(v, h->v, h->ndof * 8, kind, h->s0));
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
    CU(cudaMemcpyAsync(nhc_dev, h->nhc, h->ndof * 8 * PIMD_NHC_LENGTH, cudaMemcpyDeviceToDevice, h->s0));
    CU(cudaStreamSynchronize(h->s0));
    return PIMD_OK;
}
int pimd_set_nhc(pimd_t h, const double *nhc_dev)
{
    if (!h || !nhc_dev) return PIMD_EINVAL;
    if (h->thermostat != PIMD_THERMOSTAT_NHC) return fail(h, PIMD_EINVAL, "thermostat is not Nose-Hoover");
    int rc = ensure_ws(h);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h->nhc, nhc_dev, h->ndof * 8 * PIMD_NHC_LENGTH, cudaMemcpyDeviceToDevice, h->s0));
    return PIMD_OK;
}

static int forces_impl(pimd_t h, double *f, bool host, double *vb, int *sign)
{
    if (!h) return PIMD_EINVAL;
    int rc = eval_forces(h, true, false, 0, 0.0);
    if (rc) return rc;
    if (f) {
        double *dst = host ? h->Fout : f;
        {
            ProfScope ps(h, PIMD_PROF_COMBINE, h->s0);
            k_combine<<<(unsigned)((h->ndof + 255) / 256), 256, 0, h->s0>>>(dst, h->F, h->Fex1, h->FexP, h->ndof, h->slice, h->P);
        }
        CU(cudaGetLastError());
        if (host) CU(cudaMemcpyAsync(f, h->Fout, h->ndof * 8, cudaMemcpyDeviceToHost, h->s0));
    }
    CU(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scalars), cudaMemcpyDeviceToHost, h->s0));
    rc = read_status(h);
    if (rc) return rc;
    if (!std::isfinite(h->h_scal->vb)) return fail(h, PIMD_ENUMERIC, "V_B is not finite");
    if (vb) *vb = h->h_scal->vb;
    if (sign) *sign = h->h_scal->sign < 0 ? -1 : 1;
    return PIMD_OK;
}

static int get_forces_impl(pimd_t h, double *f, bool host)
{
    if (!h || !f) return PIMD_EINVAL;
    if (!h->forces_valid) return fail(h, PIMD_EINVAL, "no forces cached for the current positions");
    double *dst = host ? h->Fout : f;
    {
        ProfScope ps(h, PIMD_PROF_COMBINE, h->s0);
        k_combine<<<(unsigned)((h->ndof + 255) / 256), 256, 0, h->s0>>>(dst, h->F, h->Fex1, h->FexP, h->ndof, h->slice, h->P);
    }
    CU(cudaGetLastError());
    if (host) CU(cudaMemcpyAsync(f, h->Fout, h->ndof * 8, cudaMemcpyDeviceToHost, h->s0));
    CU(cudaStreamSynchronize(h->s0));
    return PIMD_OK;
}

static int set_forces_impl(pimd_t h, const double *f, cudaMemcpyKind kind)
{
    if (!h || !f) return PIMD_EINVAL;
    int rc = ensure_ws(h);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h->F, f, h->ndof * 8, kind, h->s0));
    CU(cudaMemsetAsync(h->Fex1, 0, h->slice * 8, h->s0));
    CU(cudaMemsetAsync(h->FexP, 0, h->slice * 8, h->s0));
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
    if (!h->tables_valid) return fail(h, PIMD_EINVAL, "no force evaluation to report");
    const int N = h->N;
    if (pnext) CU(cudaMemcpyAsync(pnext, h->ex.pnext, (size_t)N * 8, cudaMemcpyDeviceToHost, h->s0));
    if (vfwd || vbwd) {
        // V^{[1,n]} and V^{[u,N]} from the de-trended tables g: prefix sums of E_int and C(l,l+1)
        // are diagnostics of the evaluation, formed here in long double.
        std::vector<double> gf(2 * (size_t)(N + 1)), gb(2 * (size_t)(N + 1)), zf(N + 1), zb(N + 1), eint(N), cnext(N);
        double rf[4];
        CU(cudaMemcpyAsync(gf.data(), h->ex.g[0], (size_t)(N + 1) * 16, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(gb.data(), h->ex.g[1], (size_t)(N + 1) * 16, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(zf.data(), h->ex.gs[0], (size_t)(N + 1) * 8, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(zb.data(), h->ex.gs[1], (size_t)(N + 1) * 8, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(eint.data(), h->ex.eint, (size_t)N * 8, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(cnext.data(), h->ex.cnext, (size_t)N * 8, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaMemcpyAsync(rf, h->ex.rfin, 32, cudaMemcpyDeviceToHost, h->s0));
        CU(cudaStreamSynchronize(h->s0));
        if (h->xi == 0.0) return fail(h, PIMD_EINVAL, "tables are not formed for xi = 0");
        const long double beta = h->beta, lam = h->lambda;
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

int pimd_cycle_energies(pimd_t h, double *e_dev)
{
    if (!h || !e_dev) return PIMD_EINVAL;
    if (h->N > 65535) return fail(h, PIMD_EINVAL, "N x N output supported up to N = 65535");
    int rc = ensure_ws(h);
    if (rc) return rc;
    switch (h->d) {
    case 1: return cycle_energies_impl<1>(h, e_dev);
    case 2: return cycle_energies_impl<2>(h, e_dev);
    default: return cycle_energies_impl<3>(h, e_dev);
    }
}

int pimd_connection_probabilities(pimd_t h, double *pr_dev)
{
    if (!h || !pr_dev) return PIMD_EINVAL;
    if (h->N > 65535) return fail(h, PIMD_EINVAL, "N x N output supported up to N = 65535");
    int rc = ensure_ws(h);
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
    if (nsteps == 0) return PIMD_OK;
    int rc = ensure_ws(h);
    if (rc) return rc;
    if (!h->forces_valid) {
        rc = eval_forces(h, false, false, 0, 0.0);
        if (rc) return rc;
    }
    // open step s ; forces ; [close s + open s+1] ; forces ; ... ; close last
    rc = launch_integrate(h, false, true, 0, h->step);
    if (rc) return rc;
    int it = 0;
    const bool gauge_ok = h->gauge_valid || h->xi == 0.0;
    if (h->use_graph && !h->profiling && gauge_ok && nsteps >= 3 && ensure_graph(h) == PIMD_OK) {
        // all but the last step replay the captured graph; the step counter of the noise lives on the device meanwhile
        k_step_counter<<<1, 32, 0, h->s0>>>(h->dstep, (unsigned long long)h->step, 0);
        CU(cudaGetLastError());
        CU(cudaEventRecord(h->ev_gin, h->s0));
        CU(cudaStreamWaitEvent(h->sg, h->ev_gin, 0));
        for (; it < nsteps - 1; ++it) {
            CU(cudaGraphLaunch(h->gexec, h->sg));
            h->launches += h->graph_launches;
            h->step++;
        }
        CU(cudaEventRecord(h->ev_gout, h->sg));
        CU(cudaStreamWaitEvent(h->s0, h->ev_gout, 0));
        h->forces_valid = false; // set again below
    }
    for (; it < nsteps; ++it) {
        rc = eval_forces(h, false, false, 0, 0.0);
        if (rc) return rc;
        const bool last = it == nsteps - 1;
        rc = launch_integrate(h, true, !last, h->step, h->step + 1);
        if (rc) return rc;
        h->step++;
    }
    if (nsteps > 0) {
        // forces in F belong to the final positions: still valid
        h->forces_valid = true;
    }
    return PIMD_OK;
}

int pimd_estimators(pimd_t h, double *e_prim, double *e_vir, double *hist, int nbins, double rmax)
{
    if (!h) return PIMD_EINVAL;
    if (nbins < 0 || nbins > MAX_BINS) return fail(h, PIMD_EINVAL, "nbins must be in [0, %d]", MAX_BINS);
    if (nbins > 0 && (!hist || !(rmax > 0))) return fail(h, PIMD_EINVAL, "hist is NULL or rmax <= 0");
    int rc = eval_forces(h, true, true, nbins, rmax);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scalars), cudaMemcpyDeviceToHost, h->s0));
    CU(cudaMemcpyAsync(h->h_est, h->est, sizeof(EstAccum), cudaMemcpyDeviceToHost, h->s0));
    if (nbins > 0) CU(cudaMemcpyAsync(hist, h->hist, (size_t)nbins * 8, cudaMemcpyDeviceToHost, h->s0));
    rc = read_status(h);
    if (rc) return rc;
    // Ubar = U/P: the trap term is accumulated already divided by P, the pair terms are not
    const double ubar = h->h_est->utrap + h->h_est->upair / h->P;
    if (e_prim) *e_prim = (double)h->P * h->d * h->N / (2.0 * h->beta) - h->h_scal->ec + ubar;
    if (e_vir) *e_vir = 2.0 * h->h_est->utrap + h->h_est->virpair / h->P;
    return PIMD_OK;
}

uint64_t pimd_launch_count(pimd_t h) { return h ? h->launches : 0; }

int pimd_set_profiling(pimd_t h, int on)
{
    if (!h) return PIMD_EINVAL;
    h->profiling = on != 0;
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
