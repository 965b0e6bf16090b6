// api.cu -- the C ABI of include/poisson.h: plan creation, K^F re-layout, the 5-launch solve.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/poisson.h"
#include "generic_pass.cuh"
#include "passes.cuh"
#include "planner.hpp"
#include "registry.hpp"
#include "relayout.cuh"
#include "solve_kernel.cuh"

namespace pfft {

std::vector<KernelEntry> &kernel_registry() {
    static std::vector<KernelEntry> reg;
    return reg;
}

// Experiment knobs that may differ per pass: "n" (all five passes) or "f1,f2,f3,i2,i1".  Read at plan creation only.
static int env_pass_value(const char *name, int pass, int dflt) {
    const char *env = std::getenv(name);
    if (!env || !*env) return dflt;
    if (!std::strchr(env, ',')) return std::atoi(env);
    const char *p = env;
    for (int q = 0; q < pass && p; ++q) { p = std::strchr(p, ','); if (p) ++p; }
    return (p && *p && *p != ',') ? std::atoi(p) : dflt;
}

// variant < 0: the POISSON_VARIANT environment variable (tuning experiments; one value or one per pass), else the
// default 0.  A requested variant that was not compiled for this length falls back to variant 0.
const KernelEntry *find_kernel(int kind, int S, int pruned, int lanes_p, int prec, int variant) {
    if (variant < 0) variant = env_pass_value("POISSON_VARIANT", kind, 0);
    const KernelEntry *fallback = nullptr;
    for (const KernelEntry &e : kernel_registry())
        if (e.kind == kind && e.S == S && e.pruned == pruned && e.lanes_p == lanes_p && e.prec == prec) {
            if (e.variant == variant) return &e;
            if (e.variant == 0) fallback = &e;
        }
    return fallback;
}

// Lengths compiled in two factorizations: which one a pass takes (measured, see the inst_S*.cu file).  -1: the
// POISSON_VARIANT environment variable or the default.
static int preferred_variant(int kind, int S, int prec) {
    if (std::getenv("POISSON_VARIANT")) return -1;
    { const char *f = std::getenv("POISSON_FUSED"); if (f && f[0] == '1') return -1; }   // the fused kernel is compiled for the default factorizations
    if (S == 192 && prec == POISSON_FP64 && (kind == KIND_F2 || kind == KIND_I2)) return 9;
    return -1;
}

// ---- any-length kernel (generic_pass.cuh): a per-plan KernelEntry with run-time geometry
template <typename T>
static const void *generic_func(int kind) {
    switch (kind) {
        case KIND_F1: return reinterpret_cast<const void *>(&generic_pass_kernel<T, KIND_F1>);
        case KIND_F2: return reinterpret_cast<const void *>(&generic_pass_kernel<T, KIND_F2>);
        case KIND_F3: return reinterpret_cast<const void *>(&generic_pass_kernel<T, KIND_F3>);
        case KIND_I2: return reinterpret_cast<const void *>(&generic_pass_kernel<T, KIND_I2>);
        default: return reinterpret_cast<const void *>(&generic_pass_kernel<T, KIND_I1>);
    }
}

// Radices of S for the Stockham passes: the fewest passes over the tile with radices the kernel holds in registers
// ({2,3,4,5,6,8,10,12,14,15,16} via fft_core.cuh, 7 / 11 / 13 as written-out sums); larger radices first (their twiddle-free last
// stage is the cheapest); any other prime factor runs the one-output-per-thread fallback.
static int generic_factors(int S, int fac[16]) {
    static const int allowed[] = {16, 15, 14, 13, 12, 11, 10, 8, 7, 6, 5, 4, 3, 2};
    int n = 0, rest = S;
    // strip the prime factors the register butterflies do not cover (17 and up)
    int big[16], nbig = 0;
    {
        int r = rest;
        for (int p : {2, 3, 5, 7, 11, 13}) while (r % p == 0) r /= p;
        for (int p = 17; r > 1; p += 2) while (r % p == 0) { if (nbig == 16) return -1; big[nbig++] = p; r /= p; rest /= p; }
    }
    // fewest stages for the smooth part: depth-first over the allowed radices, non-increasing order; among equally short lists the
    // one with the smallest sum of radices (balanced radices: every stage is one sweep over the tile, whatever its radix, so a
    // radix-2 stage buys nothing -- 300 = 5 x 5 x 12 rather than 2 x 10 x 15)
    int best[16], nbest = 99, cur[16], best_sum = 1 << 30;
    struct Rec {
        static void go(int r, int start, int depth, int sum, int *cur, int *best, int &nbest, int &best_sum, const int *allowed) {
            if (r == 1) {
                if (depth < nbest || (depth == nbest && sum < best_sum)) { nbest = depth; best_sum = sum; for (int i = 0; i < depth; ++i) best[i] = cur[i]; }
                return;
            }
            if (depth + 1 > nbest || depth >= 15) return;
            for (int i = start; i < 14; ++i)
                if (r % allowed[i] == 0) { cur[depth] = allowed[i]; go(r / allowed[i], i, depth + 1, sum + allowed[i], cur, best, nbest, best_sum, allowed); }
        }
    };
    Rec::go(rest, 0, 0, 0, cur, best, nbest, best_sum, allowed);
    if (nbest == 99) return rest == 1 ? 0 : -1;
    if (nbest + nbig > 16) return -1;
    for (int i = 0; i < nbig; ++i) fac[n++] = big[i];         // the slow radices first (their pass has w_n^{jk} anyway)
    for (int i = nbest - 1; i >= 0; --i) fac[n++] = best[i];   // then ascending: the largest radix is the twiddle-free last stage
    return n;
}

static int largest_prime_factor(int S) {
    int best = 1;
    for (int p = 2; (long long)p * p <= S; ++p) while (S % p == 0) { best = p; S /= p; }
    return S > 1 ? S : best;
}

// Bluestein (generic_pass.cuh: gen_transform) for lengths with a prime factor >= 17, up to S = 1024: convolution length
// M = the smallest of {2^a, 3 2^a, 5 2^a} that is >= 2S - 1.  0: the length runs the Stockham passes directly.
static int bluestein_length(int S) {
    if (S > 1024 || largest_prime_factor(S) < 17) return 0;
    int best = 0;
    for (int base : {1, 3, 5})
        for (int m = base; m <= 4096; m *= 2)
            if (m >= 2 * S - 1) { if (!best || m < best) best = m; break; }
    return best;
}

// false: the length does not fit the any-length kernel (shared memory, or more than 16 radices)
static bool make_generic_entry(KernelEntry &e, int kind, int S, int pruned, int lanes_p, int prec) {
    e = KernelEntry{};
    e.kind = kind; e.S = S; e.pruned = pruned; e.lanes_p = lanes_p; e.prec = prec; e.generic = 1;
    e.nbuf = 2; e.NT = GEN_NT; e.TPP = 0; e.V = 0; e.RA = S; e.RB = 1;
    if (S > GEN_MAX_S) return false;
    const int M = bluestein_length(S);
    e.gen_blue = M ? 1 : 0;
    e.gen_L = M ? M : S;
    const int L = e.gen_L;
    e.gen_nfac = generic_factors(L, e.gen_fac);
    if (e.gen_nfac < 0) return false;
    const size_t cplx = prec == POISSON_FP64 ? 16 : 8;
    // widest tile (whole 128-byte rows first) that fits the 227 KB of shared memory a CTA may use
    int P = (int)(128 / cplx);
    while (P > 1 && gen_smem_bytes(L, P, cplx) > (size_t)227 * 1024) P /= 2;
    if (gen_smem_bytes(L, P, cplx) > (size_t)227 * 1024) return false;
    // two resident CTAs (16 warps) per SM matter more than whole 128-byte rows: halve the tile once if that makes room
    if (P * cplx >= 128 && gen_smem_bytes(L, P, cplx) > (size_t)112 * 1024 && gen_smem_bytes(L, P / 2, cplx) <= (size_t)112 * 1024) P /= 2;
    // small transforms: enough pencils per tile to give every thread work (L * P >= 2 * NT), still whole rows
    while (L * P < 2 * GEN_NT && P < 64 && gen_smem_bytes(L, 2 * P, cplx) <= (size_t)48 * 1024) P *= 2;
    e.P = P;
    e.smem_bytes = gen_smem_bytes(L, P, cplx);
    e.func = prec == POISSON_FP64 ? generic_func<double>(kind) : generic_func<float>(kind);
    return true;
}

std::vector<FusedEntry> &fused_registry() {
    static std::vector<FusedEntry> reg;
    return reg;
}

const FusedEntry *find_fused(int prec, const int S[3], const int pruned[3], const int lanes_p[3]) {
    for (const FusedEntry &e : fused_registry()) {
        bool same = e.prec == prec;
        for (int q = 0; q < 3 && same; ++q) same = e.S[q] == S[q] && e.pruned[q] == pruned[q] && e.lanes_p[q] == lanes_p[q];
        if (same) return &e;
    }
    return nullptr;
}

static thread_local std::string g_last_error;

static int cuda_fail(cudaError_t e, const char *what) {
    g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
    return POISSON_ECUDA;
}
#define PF_CUDA(call)                                          \
    do {                                                       \
        cudaError_t pf_e = (call);                             \
        if (pf_e != cudaSuccess) return cuda_fail(pf_e, #call); \
    } while (0)

template <typename T>
__global__ void relayout_kernel(const T *__restrict__ kuser, T *__restrict__ kint, const RelayoutParams q) {
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < q.total;
         idx += (long long)gridDim.x * blockDim.x)
        kint[idx] = relayout_value<T>(kuser, q, idx);
}

// FMA peak probe: 16 independent chains per thread, result kept alive through a never-true store.
template <typename T>
__global__ void fma_peak_kernel(T *sink, int iters, T a, T b) {
    T x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = (T)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = x[i] * a + b;
    }
    T acc = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) acc += x[i];
    if (acc == (T)123456789) sink[threadIdx.x] = acc;
}

}  // namespace pfft

using namespace pfft;

// One lane of poisson_solve_batch: its own intermediates, stream and staging, so that several solves of a
// batch are in flight at once (K^F, twiddles and kernels are shared).  Lane 0 uses the plan's own A1 / A2.
struct Lane {
    void *a1, *a2;
    void *rho_stage, *v_stage;   // host-batch staging (allocated on first use)
    cudaStream_t st;
    cudaEvent_t done;
    bool owns_ws;
    struct GraphSolve *gs;       // this lane's five launches as a CUDA graph (graph launch mode), or NULL
};

// The launches of one solve as an instantiated CUDA graph (kernel nodes F1 -> F2 -> F3 -> I2 -> I1, the middle three once per
// plane chunk): one graph launch per solve; rho / V of the call are patched into the F1 / I1 nodes when they differ from the
// previous call.
#define PF_MAX_XR 8
struct GraphSolve {
    cudaGraph_t graph;
    cudaGraphExec_t exec;
    cudaGraphNode_t node_f1, node_i1;   // the two nodes whose parameters carry rho / V of the call
    PassParams prm_f1, prm_i1;
    const void *rho;
    void *V;
    int xr;                             // > 1: F1 / I1 are split into xr kernels over ranges of x (x chains)
    cudaGraphNode_t node_f1x[PF_MAX_XR], node_i1x[PF_MAX_XR];
    PassParams prm_f1x[PF_MAX_XR], prm_i1x[PF_MAX_XR];
    long long off_rho[PF_MAX_XR], off_V[PF_MAX_XR];   // byte offsets of the ranges in rho / V
};

struct poisson_plan {
    ShardDesc *shard;          // non-NULL: plan of one rank of a sharded solve (poisson_shard_*); only those calls apply
    void *sh_mid[PF_MAX_WIDE], *sh_back[PF_MAX_WIDE];   // every rank's exchange slabs as this device addresses them
    bool sh_slabs_set;
    PlanDesc d;
    double h;
    int device;
    int num_sms;
    const KernelEntry *k[5];
    KernelEntry gen_entry[5];  // the passes that run the any-length kernel point here
    bool kcplx;                // the installed K^F is complex (poisson_set_kernel_complex)
    bool keven;                // the installed K^F is stored folded along axis b (poisson_set_kernel_even): pencils 0 .. S_b / 2 only
    int k_tpg;                 // ... in this many tiles per k_a plane
    int grid[5];
    int resident[5];      // co-resident CTAs of each pass kernel on this device
    int n_tiles[5], tiles_per_g[5];
    size_t pf_min_bytes;  // L2 prefetch (PassParams::prefetch) for arrays at least this large
    int pf_force[5];      // POISSON_PREFETCH=0..3 (one value, or one per pass) forces the prefetch bits (experiments), -1 = by size
    int chunk_planes, n_chunks; // middle passes F2 -> F3 -> I2 run chunk by chunk of k_a planes through a chunk-sized A2 (1 chunk: whole grid)
    long long a2_alloc_elems;   // complex elements of the A2 buffer actually allocated (one chunk when chunked)
    int late_tw;               // PassParams::late_tw for every pass (POISSON_LATE_TW, default 1; 0 under programmatic dependent launch)
    int pdl_trigger;           // PassParams::pdl_trigger (POISSON_PDL_TRIGGER: 0 start of the pass, 1 last tile of each CTA, 2 exit)
    bool env_shape;            // POISSON_BRANCHES / POISSON_XCHAINS given: the tuner keeps that graph shape
    int xchains;               // graph mode: F1 / F2 / I2 / I1 split over this many ranges of x (POISSON_XCHAINS)
    int branches;              // graph mode: the middle passes as this many parallel chains over ranges of k_a planes (POISSON_BRANCHES)
    int env_lanes, env_wide;   // POISSON_LANES / POISSON_WIDE as read at plan creation (-1: not set)
    int test_max_lanes;        // POISSON_TEST_MAX_LANES=n (tests only): allocating a batch lane beyond the n-th fails as if device memory had run out
    bool env_lane_graph;       // POISSON_LANE_GRAPH=0 at plan creation: plain launches on the batch lanes (experiments)
    void *wide_a1, *wide_a2;   // intermediates of wide_w densities (several small solves per launch), allocated on first use
    int wide_w;
    void *a1, *a2, *kint;
    void *tw[3];          // per axis id: exp(-2 pi i m / S) (Bluestein axes: exp(-2 pi i m / M) of the convolution length)
    void *chirp[3], *bspec[3];   // Bluestein axes only (generic_pass.cuh: gen_transform)
    void *rho_stage, *v_stage;
    const FusedEntry *fused;   // one-launch solve kernel compiled for this combination of axes, or NULL
    const FusedEntry *fused_saved; bool use_fused_saved;   // what poisson_set_kernel_even set aside (the one-launch kernel reads the full K^F layout); poisson_set_kernel puts it back
    bool use_fused;            // launch mode picked for poisson_solve: fused kernel, else 5 launches (with or without PDL)
    bool use_graph;            // ... or the five launches as one CUDA graph launch (use_pdl: with programmatic edges)
    GraphSolve gs, gs_pdl;
    float tune_ms[5];          // measured ms per solve of {5 launches, 5 launches + PDL, fused, graph, graph + PDL}; 0 = not measured
    int fused_grid, fused_skew;
    unsigned *fused_sync;      // barrier / per-plane counters of the fused kernel (zero between solves)
    size_t elem_real;     // bytes per real
    long long kint_elems;
    size_t workspace_bytes;
    bool kernel_set;
    bool use_pdl;
    std::vector<cudaEvent_t> *prof_events;  // 6 per profiled solve
    std::vector<Lane> *lanes;               // poisson_solve_batch / poisson_solve_batch_host
    cudaEvent_t fork_ev;
    int prof_count;
};

static void fill_twiddles(std::vector<unsigned char> &buf, int S, int prec) {
    const long double two_pi = 6.283185307179586476925286766559005768L;
    buf.resize((size_t)S * (prec == POISSON_FP64 ? 16 : 8));
    for (int m = 0; m < S; ++m) {
        long double c, s;
        if ((4LL * m) % S == 0) {  // exact on the axes
            const int qt = (int)((4LL * m) / S);
            c = qt == 0 ? 1.0L : (qt == 2 ? -1.0L : 0.0L);
            s = qt == 1 ? -1.0L : (qt == 3 ? 1.0L : 0.0L);
        } else {
            const long double ang = two_pi * (long double)m / (long double)S;
            c = cosl(ang); s = -sinl(ang);  // exp(-2 pi i m / S)
        }
        if (prec == POISSON_FP64) { double *o = reinterpret_cast<double *>(buf.data()) + 2 * m; o[0] = (double)c; o[1] = (double)s; }
        else { float *o = reinterpret_cast<float *>(buf.data()) + 2 * m; o[0] = (float)c; o[1] = (float)s; }
    }
}

// Bluestein tables of one axis (host, long double): chirp[n] = exp(-i pi n^2 / S), n < S (angle from n^2 mod 2S, exact), and
// bspec = DFT_M(b) / M of b[0] = 1, b[n] = b[M - n] = conj(chirp[n]) for 0 < n < S, 0 elsewhere (the 1/M of the inner inverse
// transform folded in).  The DFT is the O(M^2) definition: M <= 2048, a few tens of milliseconds once per plan.
static void fill_bluestein(std::vector<unsigned char> &chirp, std::vector<unsigned char> &bspec, int S, int M, int prec) {
    const long double pi = 3.141592653589793238462643383279502884L;
    std::vector<long double> cr(S), ci(S), br(M, 0.0L), bi(M, 0.0L);
    for (int n = 0; n < S; ++n) {
        const long long m = ((long long)n * n) % (2LL * S);
        const long double ang = pi * (long double)m / (long double)S;
        cr[n] = cosl(ang); ci[n] = -sinl(ang);
        br[n] = cr[n]; bi[n] = -ci[n];
        if (n) { br[M - n] = br[n]; bi[M - n] = bi[n]; }
    }
    std::vector<long double> wr(M), wi(M);
    for (int m = 0; m < M; ++m) { const long double a = 2.0L * pi * (long double)m / (long double)M; wr[m] = cosl(a); wi[m] = -sinl(a); }
    const size_t el = prec == POISSON_FP64 ? 16 : 8;
    chirp.resize((size_t)S * el); bspec.resize((size_t)M * el);
    auto put = [&](std::vector<unsigned char> &buf, int i, long double re, long double im) {
        if (prec == POISSON_FP64) { double *o = reinterpret_cast<double *>(buf.data()) + 2 * i; o[0] = (double)re; o[1] = (double)im; }
        else { float *o = reinterpret_cast<float *>(buf.data()) + 2 * i; o[0] = (float)re; o[1] = (float)im; }
    };
    for (int n = 0; n < S; ++n) put(chirp, n, cr[n], ci[n]);
    for (int k = 0; k < M; ++k) {
        long double sr = 0.0L, si = 0.0L;
        long long idx = 0;
        for (int n = 0; n < M; ++n) {
            if (br[n] != 0.0L || bi[n] != 0.0L) { sr += br[n] * wr[idx] - bi[n] * wi[idx]; si += br[n] * wi[idx] + bi[n] * wr[idx]; }
            idx += k; if (idx >= M) idx -= M;
        }
        put(bspec, k, sr / M, si / M);
    }
}

static void free_plan(poisson_plan *pl) {
    if (!pl) return;
    delete pl->shard;
    cudaFree(pl->a1); cudaFree(pl->a2); cudaFree(pl->kint);
    for (int q = 0; q < 3; ++q) { cudaFree(pl->tw[q]); cudaFree(pl->chirp[q]); cudaFree(pl->bspec[q]); }
    cudaFree(pl->rho_stage); cudaFree(pl->v_stage); cudaFree(pl->fused_sync);
    cudaFree(pl->wide_a1); cudaFree(pl->wide_a2);
    for (GraphSolve *g : {&pl->gs, &pl->gs_pdl}) { if (g->exec) cudaGraphExecDestroy(g->exec); if (g->graph) cudaGraphDestroy(g->graph); }
    if (pl->lanes) {
        for (Lane &ln : *pl->lanes) {
            if (ln.owns_ws) { cudaFree(ln.a1); cudaFree(ln.a2); }
            if (ln.gs) { if (ln.gs->exec) cudaGraphExecDestroy(ln.gs->exec); if (ln.gs->graph) cudaGraphDestroy(ln.gs->graph); delete ln.gs; }
            cudaFree(ln.rho_stage); cudaFree(ln.v_stage);
            if (ln.st) cudaStreamDestroy(ln.st);
            if (ln.done) cudaEventDestroy(ln.done);
        }
        delete pl->lanes;
    }
    if (pl->fork_ev) cudaEventDestroy(pl->fork_ev);
    if (pl->prof_events) {
        for (cudaEvent_t e : *pl->prof_events) cudaEventDestroy(e);
        delete pl->prof_events;
    }
    delete pl;
}

static int check_device(const poisson_plan *pl, bool want_shard = false) {
    if ((pl->shard != nullptr) != want_shard) {
        g_last_error = want_shard ? "not a shard plan (poisson_shard_plan_create)" : "a shard plan only takes the poisson_shard_* calls";
        return POISSON_EINVAL;
    }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != pl->device) {
        cudaGetLastError();
        g_last_error = "the current CUDA device is not the one the plan was created on";
        return POISSON_EINVAL;
    }
    return POISSON_OK;
}

static GraphSolve *active_graph(poisson_plan *pl) {
    GraphSolve *g = pl->use_pdl ? &pl->gs_pdl : &pl->gs;
    return g->exec ? g : nullptr;
}
static const GraphSolve *active_graph(const poisson_plan *pl) { return active_graph(const_cast<poisson_plan *>(pl)); }

static int launches_per_solve(const poisson_plan *pl) { return pl->n_chunks <= 1 ? 5 : 2 + 3 * pl->n_chunks; }

// Reals in the internal K^F copy: the register-engine F3 streams [tile][V][NT] (padded to whole tiles), the any-length
// kernel reads the natural order of the pass (one real, or one complex number, per spectrum point).
static long long kint_reals(const poisson_plan *pl) {
    const KernelEntry *e = pl->k[2];
    if (e->generic) return (long long)pl->d.pass[2].n_g * pl->d.pass[2].S * pl->d.pass[2].n_p * (pl->kcplx ? 2 : 1);
    if (pl->keven) return (long long)pl->d.pass[2].n_g * pl->k_tpg * e->V * e->NT;
    return (long long)pl->n_tiles[2] * e->V * e->NT;
}

// Plane chunks for the middle passes (see for_each_launch).  OPT-IN: measured on B200 the chunked 512^3 solve moves 1.9 GB
// instead of 4.0 GB through HBM and shrinks the workspace by most of A2, but it is SLOWER (fp64 794 -> 863 us with 96 MB
// chunks, 910 us with 64 MB, 1111 us with 32 MB; fp32 449 -> 467 us): the S = 512 passes are held by their FP64 / shared-memory
// pipes at 8 warps per SM, not by DRAM, and every extra launch costs a ramp-up and a partly filled last wave (DESIGN.md
// section 10).  POISSON_CHUNK=n: n planes per chunk; POISSON_CHUNK_MB=m: chunks of about m MB, sized within [m/2, m] to the
// plane count that leaves the smallest partly-filled last wave of tiles in the three middle passes.
static void choose_chunks(poisson_plan *pl) {
    const PlanDesc &d = pl->d;
    const size_t cplx = 2 * pl->elem_real;
    const long long plane_elems = d.a2_elems / d.H;
    pl->chunk_planes = d.H; pl->n_chunks = 1; pl->a2_alloc_elems = d.a2_elems;
    const char *env = std::getenv("POISSON_CHUNK");
    const char *env_mb = std::getenv("POISSON_CHUNK_MB");
    int planes = 0;
    if (env) planes = std::atoi(env);
    else if (env_mb && std::atof(env_mb) > 0.0) {
        const double target = std::atof(env_mb) * 1048576.0;
        const int pmax = (int)(target / ((double)plane_elems * cplx));
        double best = -1.0;
        for (int p = pmax; p >= 1 && p >= pmax / 2; --p) {
            double eff = 1.0;
            for (int q = POISSON_PASS_F2; q <= POISSON_PASS_I2; ++q) {
                const long long T = (long long)p * pl->tiles_per_g[q], R = pl->resident[q];
                const double e = (double)T / (double)(((T + R - 1) / R) * R);
                eff = e < eff ? e : eff;
            }
            if (eff > best + 1e-9) { best = eff; planes = p; }
        }
    }
    if (planes >= 1 && planes < d.H) {
        pl->chunk_planes = planes;
        pl->n_chunks = (d.H + planes - 1) / planes;
        pl->a2_alloc_elems = plane_elems * planes;
    }
}

// Picks the kernel of pass q (the compiled register-engine kernel for its length, else -- or when force_generic -- the
// any-length kernel) and derives tiles, occupancy and the persistent grid from it.
static int setup_pass(poisson_plan *pl, int q, bool force_generic) {
    const PassDesc &ps = pl->d.pass[q];
    const int precision = pl->d.prec;
    const KernelEntry *e = nullptr;
    if (!ps.generic && !force_generic)
        e = find_kernel(ps.kind, ps.S, ps.pruned, ps.lanes_p, precision, preferred_variant(ps.kind, ps.S, precision));
    if (!e) {
        // F1 / I1 address rho / V in pairs (register engine) or in reals (any-length kernel): the planner fixed which
        if (!ps.generic && (q == POISSON_PASS_F1 || q == POISSON_PASS_I1)) return POISSON_EUNSUPPORTED;
        if (!make_generic_entry(pl->gen_entry[q], ps.kind, ps.S, ps.pruned, ps.lanes_p, precision)) return POISSON_EUNSUPPORTED;
        e = &pl->gen_entry[q];
    }
    pl->k[q] = e;
    pl->tiles_per_g[q] = (int)((ps.n_p + e->P - 1) / e->P);
    pl->n_tiles[q] = (int)(ps.n_g * pl->tiles_per_g[q]);
    cudaError_t ce = cudaFuncSetAttribute(e->func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)e->smem_bytes);
    if (ce != cudaSuccess) return cuda_fail(ce, "cudaFuncSetAttribute(smem)");
    int occ = 0;
    ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, e->func, e->NT, e->smem_bytes);
    if (ce != cudaSuccess || occ < 1) return cuda_fail(ce, "occupancy query");
    const long long resident = (long long)occ * pl->num_sms;
    pl->resident[q] = (int)resident;
    pl->grid[q] = (int)(pl->n_tiles[q] < resident ? pl->n_tiles[q] : resident);  // persistent CTAs
    { const int force = env_pass_value("POISSON_GRID", q, 0);                     // experiments: CTAs of pass q
      if (force > 0 && force < pl->grid[q]) pl->grid[q] = force; }
    return POISSON_OK;
}

extern "C" {

static int tune_plan(poisson_plan *pl);

const char *poisson_status_string(int st) {
    switch (st) {
        case POISSON_OK: return "ok";
        case POISSON_EINVAL: return "invalid argument";
        case POISSON_EUNSUPPORTED: return "unsupported grid size (a padded length above the any-length kernel's limit of 4096)";
        case POISSON_ENOMEM: return "out of memory";
        case POISSON_ENOKERNEL: return "poisson_solve called before poisson_set_kernel";
        case POISSON_ECUDA: return "CUDA error (see poisson_last_error)";
        case POISSON_EARCH: return "no CUDA device of compute capability 10.x (kernels are built for sm_100a)";
        default: return "unknown status";
    }
}

const char *poisson_last_error(void) { return g_last_error.c_str(); }

const char *poisson_build_arch(void) { return "sm_100a"; }

int poisson_plan_describe(int nx, int ny, int nz, const int bc[3], int precision, poisson_plan_info *info) {
    if (!info) return POISSON_EINVAL;
    PlanDesc d;
    const int st = plan_build(nx, ny, nz, bc, precision, d);
    if (st != POISSON_OK) return st;
    for (int q = 0; q < 5; ++q) {
        const PassDesc &ps = d.pass[q];
        KernelEntry tmp;
        if (!ps.generic && find_kernel(ps.kind, ps.S, ps.pruned, ps.lanes_p, precision)) continue;
        if (!ps.generic && (q == POISSON_PASS_F1 || q == POISSON_PASS_I1)) return POISSON_EUNSUPPORTED;
        if (!make_generic_entry(tmp, ps.kind, ps.S, ps.pruned, ps.lanes_p, precision)) return POISSON_EUNSUPPORTED;
    }
    *info = d.info;
    return POISSON_OK;
}

int poisson_plan_create(poisson_plan **out, int nx, int ny, int nz, const int bc[3], double h, int precision) {
    if (!out) return POISSON_EINVAL;
    *out = nullptr;
    if (!(h > 0.0) || !std::isfinite(h)) return POISSON_EINVAL;
    PlanDesc d;
    int st = plan_build(nx, ny, nz, bc, precision, d);
    if (st != POISSON_OK) return st;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        g_last_error = "no CUDA device";
        return POISSON_EARCH;
    }
    int dev = 0;
    PF_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    PF_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) {
        g_last_error = "device is sm_" + std::to_string(prop.major * 10 + prop.minor) + ", kernels are sm_100a";
        return POISSON_EARCH;
    }

    poisson_plan *pl = new (std::nothrow) poisson_plan();
    if (!pl) return POISSON_ENOMEM;
    std::memset(static_cast<void *>(pl), 0, sizeof(*pl));
    pl->d = d; pl->h = h; pl->device = dev; pl->num_sms = prop.multiProcessorCount;
    pl->elem_real = precision == POISSON_FP64 ? 8 : 4;
    // Programmatic dependent launch is opt-in (POISSON_PDL=1): measured on B200 it shortens back-to-back
    // launches of one pass but lengthens the 5-pass solve ("What was tried").
    // Launch mode: five launches, five launches with programmatic dependent launch, or the one-launch fused
    // kernel.  Which is fastest depends on the grid (PDL wins on launch-bound grids), so
    // poisson_plan_create MEASURES the candidates once (tune_plan below) unless POISSON_TUNE=0 or the mode is
    // forced with POISSON_PDL=0|1 / POISSON_FUSED=0|1.
    { const char *env = std::getenv("POISSON_PDL"); pl->use_pdl = env && env[0] == '1'; }
    for (int q = 0; q < 5; ++q) pl->pf_force[q] = env_pass_value("POISSON_PREFETCH", q, -1);
    // every environment knob is read HERE, once; the solve path never calls getenv
    { const char *env = std::getenv("POISSON_LATE_TW"); pl->late_tw = env ? std::atoi(env) : 1; }
    { const char *env = std::getenv("POISSON_PDL_TRIGGER"); pl->pdl_trigger = env ? std::atoi(env) : 1; }
    { const char *env = std::getenv("POISSON_BRANCHES"); pl->branches = env ? std::atoi(env) : 1; }
    { const char *env = std::getenv("POISSON_XCHAINS"); pl->xchains = env ? std::atoi(env) : 1; if (pl->xchains > PF_MAX_XR) pl->xchains = PF_MAX_XR; }
    pl->env_shape = std::getenv("POISSON_BRANCHES") || std::getenv("POISSON_XCHAINS");
    { const char *env = std::getenv("POISSON_LANES"); pl->env_lanes = env ? std::atoi(env) : -1; }
    { const char *env = std::getenv("POISSON_WIDE"); pl->env_wide = env ? std::atoi(env) : -1; }
    { const char *env = std::getenv("POISSON_LANE_GRAPH"); pl->env_lane_graph = !(env && env[0] == '0'); }
    { const char *env = std::getenv("POISSON_TEST_MAX_LANES"); pl->test_max_lanes = env ? std::atoi(env) : 0; }
    pl->pf_min_bytes = (size_t)96 << 20;

    for (int q = 0; q < 5; ++q) {
        st = setup_pass(pl, q, false);
        if (st != POISSON_OK) { free_plan(pl); return st; }
    }

    choose_chunks(pl);

    // One-launch fused solve (solve_kernel.cuh) when this combination of axes was compiled and the per-pass
    // tiles agree with it; POISSON_FUSED=0 keeps the 5-launch path (per-pass experiments).
    {
        const char *env = std::getenv("POISSON_FUSED");
        const bool want = !(env && env[0] == '0');
        pl->use_fused = env && env[0] == '1';
        int S3[3], pr3[3], lp3[3];
        const int qs[3] = {POISSON_PASS_F1, POISSON_PASS_F2, POISSON_PASS_F3};
        for (int q = 0; q < 3; ++q) { S3[q] = d.pass[qs[q]].S; pr3[q] = d.pass[qs[q]].pruned; lp3[q] = d.pass[qs[q]].lanes_p; }
        const FusedEntry *fe = (want && pl->n_chunks <= 1) ? find_fused(precision, S3, pr3, lp3) : nullptr;   // the fused kernel needs all of A2
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        bool any_generic = false;
        for (int q = 0; q < 5; ++q) any_generic = any_generic || pl->k[q]->generic;
        if (fe && coop && !any_generic && fe->P[0] == pl->k[0]->P && fe->P[1] == pl->k[1]->P && fe->P[2] == pl->k[2]->P &&
            d.pass[1].n_g == d.H && d.pass[2].n_g == d.H) {
            cudaError_t ce = cudaFuncSetAttribute(fe->func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fe->smem_bytes);
            int occ = 0;
            if (ce == cudaSuccess) ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fe->func, fe->NT, fe->smem_bytes);
            if (ce != cudaSuccess || occ < 1) { free_plan(pl); return cuda_fail(ce, "fused kernel occupancy query"); }
            const long long resident = (long long)occ * pl->num_sms;
            const long long per_step = 2LL * pl->tiles_per_g[1] + pl->tiles_per_g[2];
            long long most = (long long)d.H * per_step;
            if (pl->n_tiles[0] > most) most = pl->n_tiles[0];
            pl->fused = fe;
            pl->fused_grid = (int)(most < resident ? most : resident);
            // skew D: the first D steps hold F2 tiles only and the last D steps I2 tiles only, so D * T2 >= grid
            // keeps every CTA busy through ramp-up and drain; it also puts a plane's F3 items several rounds
            // behind its F2 items, so the per-plane waits are (almost) never taken
            { const char *envd = std::getenv("POISSON_FUSED_SKEW");
              pl->fused_skew = envd ? std::atoi(envd) : (pl->fused_grid + pl->tiles_per_g[1] - 1) / pl->tiles_per_g[1] + 1;
              if (pl->fused_skew < 1) pl->fused_skew = 1; }
            const size_t sync_bytes = (size_t)(2 + 2 * d.H) * sizeof(unsigned);
            ce = cudaMalloc(reinterpret_cast<void **>(&pl->fused_sync), sync_bytes);
            if (ce == cudaSuccess) ce = cudaMemset(pl->fused_sync, 0, sync_bytes);
            if (ce != cudaSuccess) { free_plan(pl); return cuda_fail(ce, "fused kernel counters"); }
        }
    }

    const size_t cplx = 2 * pl->elem_real;
    pl->kint_elems = kint_reals(pl);
    size_t ws = 0;
    cudaError_t ce = cudaMalloc(&pl->a1, (size_t)d.a1_elems * cplx); ws += (size_t)d.a1_elems * cplx;
    if (ce == cudaSuccess) { ce = cudaMalloc(&pl->a2, (size_t)pl->a2_alloc_elems * cplx); ws += (size_t)pl->a2_alloc_elems * cplx; }
    if (ce == cudaSuccess) { ce = cudaMalloc(&pl->kint, (size_t)pl->kint_elems * pl->elem_real); ws += (size_t)pl->kint_elems * pl->elem_real; }
    for (int q = 0; q < 3 && ce == cudaSuccess; ++q) {
        // a Bluestein axis (all passes of an axis agree: same length, any-length kernel) carries the table of its
        // convolution length M plus the chirp and its spectrum
        int M = 0;
        for (int ps = 0; ps < 5; ++ps) if (d.pass[ps].axis == q && pl->k[ps]->generic && pl->k[ps]->gen_blue) M = pl->k[ps]->gen_L;
        std::vector<unsigned char> host;
        fill_twiddles(host, M ? M : d.s[q], precision);
        ce = cudaMalloc(&pl->tw[q], host.size());
        if (ce == cudaSuccess) ce = cudaMemcpy(pl->tw[q], host.data(), host.size(), cudaMemcpyHostToDevice);
        ws += host.size();
        if (M && ce == cudaSuccess) {
            std::vector<unsigned char> hc, hb;
            fill_bluestein(hc, hb, d.s[q], M, precision);
            ce = cudaMalloc(&pl->chirp[q], hc.size());
            if (ce == cudaSuccess) ce = cudaMemcpy(pl->chirp[q], hc.data(), hc.size(), cudaMemcpyHostToDevice);
            if (ce == cudaSuccess) ce = cudaMalloc(&pl->bspec[q], hb.size());
            if (ce == cudaSuccess) ce = cudaMemcpy(pl->bspec[q], hb.data(), hb.size(), cudaMemcpyHostToDevice);
            ws += hc.size() + hb.size();
        }
    }
    if (ce != cudaSuccess) {
        free_plan(pl);
        if (ce == cudaErrorMemoryAllocation) { cudaGetLastError(); return POISSON_ENOMEM; }
        return cuda_fail(ce, "workspace allocation");
    }
    pl->workspace_bytes = ws;
    pl->d.info.workspace_bytes = (long long)ws;
    st = tune_plan(pl);
    if (st != POISSON_OK) { free_plan(pl); return st; }
    *out = pl;
    return POISSON_OK;
}

int poisson_measure_fma_peak(int precision, double *tflops) {
    if (!tflops || (precision != POISSON_FP64 && precision != POISSON_FP32)) return POISSON_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return POISSON_EARCH; }
    int dev = 0;
    PF_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    PF_CUDA(cudaGetDeviceProperties(&prop, dev));
    void *sink = nullptr;
    PF_CUDA(cudaMalloc(&sink, 1024 * sizeof(double)));
    cudaEvent_t e0, e1;
    PF_CUDA(cudaEventCreate(&e0));
    PF_CUDA(cudaEventCreate(&e1));
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 4096;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        PF_CUDA(cudaEventRecord(e0));
        if (precision == POISSON_FP64) fma_peak_kernel<double><<<blocks, threads>>>(static_cast<double *>(sink), iters, 1.0000001, 1e-9);
        else fma_peak_kernel<float><<<blocks, threads>>>(static_cast<float *>(sink), iters, 1.0000001f, 1e-9f);
        PF_CUDA(cudaEventRecord(e1));
        PF_CUDA(cudaEventSynchronize(e1));
        float ms = 0.f;
        PF_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    const double flops = 2.0 * 16.0 * (double)iters * (double)blocks * (double)threads;
    *tflops = flops / (best_ms * 1e-3) / 1e12;
    return POISSON_OK;
}

int poisson_plan_kernel_dims(const poisson_plan *pl, long long dims[3]) {
    if (!pl || !dims) return POISSON_EINVAL;
    dims[0] = pl->d.s[2]; dims[1] = pl->d.s[1]; dims[2] = pl->d.s[0] / 2 + 1;
    return POISSON_OK;
}

int poisson_plan_get_info(const poisson_plan *pl, poisson_plan_info *info) {
    if (!pl || !info) return POISSON_EINVAL;
    *info = pl->d.info;
    return POISSON_OK;
}

size_t poisson_plan_workspace_bytes(const poisson_plan *pl) { return pl ? pl->workspace_bytes : 0; }

// kernels per solve (graph mode: that many kernel nodes; a shaped graph has R F1 + R J F2 + J F3 + R J I2 + R I1 of them)
int poisson_plan_launches_per_solve(const poisson_plan *pl) {
    if (!pl) return 0;
    if (pl->fused && pl->use_fused) return 1;
    int J = 1, R = 1;
    if (poisson_plan_graph_shape(pl, &J, &R) == POISSON_OK && (J > 1 || R > 1)) return 2 * R + 2 * R * J + J;
    return launches_per_solve(pl);
}

int poisson_plan_launch_mode(const poisson_plan *pl, int *mode, double ms_per_solve[5]) {
    if (!pl || !mode || !ms_per_solve) return POISSON_EINVAL;
    *mode = pl->fused && pl->use_fused ? POISSON_LAUNCH_FUSED
          : (pl->use_graph && active_graph(pl) ? (pl->use_pdl ? POISSON_LAUNCH_GRAPH_PDL : POISSON_LAUNCH_GRAPH)
                                               : (pl->use_pdl ? POISSON_LAUNCH_FIVE_PDL : POISSON_LAUNCH_FIVE));
    for (int m = 0; m < 5; ++m) ms_per_solve[m] = (double)pl->tune_ms[m];
    return POISSON_OK;
}

int poisson_plan_graph_shape(const poisson_plan *pl, int *plane_chains, int *x_chains) {
    if (!pl || !plane_chains || !x_chains) return POISSON_EINVAL;
    const GraphSolve *g = (pl->use_graph && !(pl->fused && pl->use_fused)) ? active_graph(pl) : nullptr;
    *plane_chains = g && pl->n_chunks <= 1 && pl->branches > 1 ? (pl->branches < pl->d.H ? pl->branches : pl->d.H) : 1;
    *x_chains = g && g->xr > 1 ? g->xr : 1;
    return POISSON_OK;
}

int poisson_plan_destroy(poisson_plan *pl) {
    if (!pl) return POISSON_EINVAL;
    free_plan(pl);
    return POISSON_OK;
}

static void destroy_graph(GraphSolve &g) {
    if (g.exec) cudaGraphExecDestroy(g.exec);
    if (g.graph) cudaGraphDestroy(g.graph);
    std::memset(&g, 0, sizeof(g));
}

static int build_graph(poisson_plan *pl, GraphSolve &g, const Lane *ln);
static int build_graph_pdl(poisson_plan *pl, GraphSolve &g, const Lane *ln);

// Re-lays the caller's K^F into the order pass F3 consumes it, for either F3 kernel.
static int relayout_kernel_spectrum(poisson_plan *pl, const void *K_f_dev, bool cplx, cudaStream_t st) {
    const PlanDesc &d = pl->d;
    const KernelEntry *e = pl->k[2];
    const double scale = 1.0 / ((double)d.s[0] * (double)d.s[1] * (double)d.s[2]);  // reading 2: one 1/(SxSySz)
    const int threads = 256;
    if (e->generic) {
        GenericRelayoutParams q;
        q.S = d.pass[2].S; q.n_p = (int)d.pass[2].n_p; q.lanes_p = d.pass[2].lanes_p; q.cplx = cplx ? 1 : 0;
        q.a_axis = d.order[0]; q.c_axis = d.order[2];
        q.sx = d.s[0]; q.sy = d.s[1]; q.sz = d.s[2];
        q.total = (long long)d.pass[2].n_g * q.S * q.n_p;
        q.scale = scale;
        long long blocks = (q.total + threads - 1) / threads;
        if (blocks > 148LL * 32) blocks = 148LL * 32;
        if (d.prec == POISSON_FP64)
            generic_relayout_kernel<double><<<(int)blocks, threads, 0, st>>>(static_cast<const double *>(K_f_dev), static_cast<double *>(pl->kint), q);
        else
            generic_relayout_kernel<float><<<(int)blocks, threads, 0, st>>>(static_cast<const float *>(K_f_dev), static_cast<float *>(pl->kint), q);
    } else {
        RelayoutParams q;
        q.g0 = pl->shard ? pl->shard->k0 : 0;
        q.RA = e->RA; q.RB = e->RB; q.TPP = e->TPP; q.P = e->P; q.V = e->V; q.NT = e->NT; q.lanes_p = e->lanes_p;
        q.tiles_per_g = pl->keven ? pl->k_tpg : pl->tiles_per_g[2]; q.n_p = (int)d.pass[2].n_p;
        q.fold = pl->keven ? (int)d.pass[2].n_p : 0;
        q.a_axis = d.order[0]; q.c_axis = d.order[2];
        q.sx = d.s[0]; q.sy = d.s[1]; q.sz = d.s[2];
        q.total = pl->kint_elems;
        q.scale = scale;
        long long blocks = (q.total + threads - 1) / threads;
        if (blocks > 148LL * 32) blocks = 148LL * 32;
        if (d.prec == POISSON_FP64)
            relayout_kernel<double><<<(int)blocks, threads, 0, st>>>(static_cast<const double *>(K_f_dev), static_cast<double *>(pl->kint), q);
        else
            relayout_kernel<float><<<(int)blocks, threads, 0, st>>>(static_cast<const float *>(K_f_dev), static_cast<float *>(pl->kint), q);
    }
    PF_CUDA(cudaGetLastError());
    return POISSON_OK;
}

// Switches the internal K^F copy between the full and the folded layout (poisson_set_kernel_even): the buffer is re-allocated at
// its new size and everything built around pass F3's parameters (graphs, the one-launch kernel's addressing) is dropped / rebuilt.
static int switch_kernel_fold(poisson_plan *pl, bool even) {
    if (pl->keven == even) return POISSON_OK;
    PF_CUDA(cudaDeviceSynchronize());   // no solve of this plan may still be reading the buffer replaced below
    const bool was = pl->keven;
    pl->keven = even;
    pl->k_tpg = (int)((pl->d.pass[2].n_p / 2 + 1 + pl->k[2]->P - 1) / pl->k[2]->P);
    const long long need = kint_reals(pl);
    void *fresh = nullptr;
    cudaError_t ce = cudaMalloc(&fresh, (size_t)need * pl->elem_real);
    if (ce != cudaSuccess) { cudaGetLastError(); pl->keven = was; return ce == cudaErrorMemoryAllocation ? POISSON_ENOMEM : cuda_fail(ce, "K^F allocation"); }
    cudaFree(pl->kint);
    pl->kint = fresh;
    pl->workspace_bytes += (size_t)need * pl->elem_real;
    pl->workspace_bytes -= (size_t)pl->kint_elems * pl->elem_real;
    pl->d.info.workspace_bytes = (long long)pl->workspace_bytes;
    pl->kint_elems = need;
    pl->kernel_set = false;
    destroy_graph(pl->gs); destroy_graph(pl->gs_pdl);
    if (pl->lanes) for (Lane &ln : *pl->lanes) if (ln.gs) destroy_graph(*ln.gs);
    if (even) {   // the one-launch kernel addresses the full layout: set it (and the tuned choice) aside while the copy is folded
        pl->fused_saved = pl->fused; pl->use_fused_saved = pl->use_fused;
        pl->fused = nullptr; pl->use_fused = false;
    } else if (pl->fused_saved) {
        pl->fused = pl->fused_saved; pl->use_fused = pl->use_fused_saved;
        pl->fused_saved = nullptr;
    }
    if (pl->use_graph) { if ((pl->use_pdl ? build_graph_pdl(pl, pl->gs_pdl, nullptr) : build_graph(pl, pl->gs, nullptr)) != POISSON_OK) cudaGetLastError(); }
    return POISSON_OK;
}

int poisson_set_kernel_even(poisson_plan *pl, const void *K_f_dev, void *stream) {
    if (!pl || !K_f_dev) return POISSON_EINVAL;
    if (reinterpret_cast<size_t>(K_f_dev) % 16) return POISSON_EINVAL;
    if (check_device(pl) != POISSON_OK) return POISSON_EINVAL;
    if (pl->k[2]->generic || pl->kcplx) return POISSON_EUNSUPPORTED;   // the register-engine F3 kernels only
    int rc = switch_kernel_fold(pl, true);
    if (rc != POISSON_OK) return rc;
    rc = relayout_kernel_spectrum(pl, K_f_dev, false, reinterpret_cast<cudaStream_t>(stream));
    if (rc != POISSON_OK) return rc;
    pl->kernel_set = true;
    return POISSON_OK;
}

int poisson_set_kernel(poisson_plan *pl, const void *K_f_dev, void *stream) {
    if (!pl || !K_f_dev) return POISSON_EINVAL;
    if (reinterpret_cast<size_t>(K_f_dev) % 16) return POISSON_EINVAL;
    if (check_device(pl) != POISSON_OK) return POISSON_EINVAL;
    if (pl->keven) { const int rc0 = switch_kernel_fold(pl, false); if (rc0 != POISSON_OK) return rc0; }
    if (pl->kcplx) {   // back from a complex kernel: the any-length F3 kernel stays, its K^F copy holds reals again
        pl->kcplx = false;
        destroy_graph(pl->gs); destroy_graph(pl->gs_pdl);
        if (pl->lanes) for (Lane &ln : *pl->lanes) if (ln.gs) destroy_graph(*ln.gs);
        if (pl->use_graph) { if ((pl->use_pdl ? build_graph_pdl(pl, pl->gs_pdl, nullptr) : build_graph(pl, pl->gs, nullptr)) != POISSON_OK) cudaGetLastError(); }
    }
    const int rc = relayout_kernel_spectrum(pl, K_f_dev, false, reinterpret_cast<cudaStream_t>(stream));
    if (rc != POISSON_OK) return rc;
    pl->kernel_set = true;
    return POISSON_OK;
}

int poisson_set_kernel_complex(poisson_plan *pl, const void *K_f_dev, void *stream) {
    if (!pl || !K_f_dev) return POISSON_EINVAL;
    if (reinterpret_cast<size_t>(K_f_dev) % 16) return POISSON_EINVAL;
    if (check_device(pl) != POISSON_OK) return POISSON_EINVAL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (pl->keven) { const int rc0 = switch_kernel_fold(pl, false); if (rc0 != POISSON_OK) return rc0; }
    if (!pl->kcplx) {
        // The complex multiply lives in the any-length F3 kernel: switch pass F3 to it (once), drop what was built
        // around the old kernel (graphs, the fused one-launch kernel), and size the internal K^F copy for complex values.
        PF_CUDA(cudaDeviceSynchronize());   // no solve of this plan may still be using the buffers replaced below
        destroy_graph(pl->gs); destroy_graph(pl->gs_pdl);
        if (pl->lanes) for (Lane &ln : *pl->lanes) if (ln.gs) destroy_graph(*ln.gs);
        pl->fused = nullptr; pl->use_fused = false; pl->fused_saved = nullptr;   // for good: pass F3 leaves the register engine
        if (!pl->k[2]->generic) { const int rc = setup_pass(pl, 2, true); if (rc != POISSON_OK) return rc; }
        pl->kcplx = true;
        const long long need = kint_reals(pl);
        if (need > pl->kint_elems) {
            void *fresh = nullptr;
            cudaError_t ce = cudaMalloc(&fresh, (size_t)need * pl->elem_real);
            if (ce != cudaSuccess) { cudaGetLastError(); pl->kcplx = false; return ce == cudaErrorMemoryAllocation ? POISSON_ENOMEM : cuda_fail(ce, "complex K^F allocation"); }
            cudaFree(pl->kint);
            pl->kint = fresh;
            pl->workspace_bytes += (size_t)(need - pl->kint_elems) * pl->elem_real;
            pl->kint_elems = need;
        }
        pl->kernel_set = false;
        if (pl->use_graph) { if ((pl->use_pdl ? build_graph_pdl(pl, pl->gs_pdl, nullptr) : build_graph(pl, pl->gs, nullptr)) != POISSON_OK) cudaGetLastError(); }
    }
    const int rc = relayout_kernel_spectrum(pl, K_f_dev, true, st);
    if (rc != POISSON_OK) return rc;
    pl->kernel_set = true;
    return POISSON_OK;
}

static PassParams pass_params(const poisson_plan *pl, int q, const void *rho, void *V, const Lane *ln = nullptr) {
    const PassDesc &ps = pl->d.pass[q];
    void *a1 = ln ? ln->a1 : pl->a1, *a2 = ln ? ln->a2 : pl->a2;
    PassParams prm{};
    switch (q) {
        case POISSON_PASS_F1: prm.in = rho; prm.out = a1; break;
        case POISSON_PASS_F2: prm.in = a1; prm.out = a2; break;
        case POISSON_PASS_F3: prm.in = a2; prm.out = a2; break;
        case POISSON_PASS_I2: prm.in = a2; prm.out = a1; break;
        default: prm.in = a1; prm.out = V; break;
    }
    prm.kint = pl->kint;
    if (q == POISSON_PASS_F3 && pl->keven) { prm.k_fold = (int)ps.n_p; prm.k_tpg = pl->k_tpg; }
    prm.tw = pl->tw[ps.axis];
    prm.gs_in = ps.gs_in; prm.ns_in = ps.ns_in; prm.ps_in = ps.ps_in;
    prm.gs_out = ps.gs_out; prm.ns_out = ps.ns_out; prm.ps_out = ps.ps_out;
    prm.n_p = (int)ps.n_p; prm.tiles_per_g = pl->tiles_per_g[q]; prm.n_tiles = pl->n_tiles[q];
    prm.n_tiles1 = pl->n_tiles[q];   // one density per launch
    // twiddle tables under the first tile's load latency; with programmatic dependent launch they are built BEFORE the wait
    // on the previous pass instead (that is the part of a pass PDL overlaps with its predecessor's tail)
    prm.late_tw = (pl->late_tw == 2 || (pl->late_tw && !pl->use_pdl)) ? 1 : 0;   // POISSON_LATE_TW=2: late also under PDL (experiments)
    prm.pdl_trigger = pl->pdl_trigger;
    if (pl->k[q]->generic) {
        const KernelEntry *e = pl->k[q];
        prm.gen_S = e->S; prm.gen_P = e->P; prm.gen_nfac = e->gen_nfac; prm.gen_pruned = e->pruned;
        prm.gen_nreal = ps.n_real; prm.gen_kcplx = pl->kcplx ? 1 : 0; prm.gen_lanes_p = ps.lanes_p;
        prm.gen_L = e->gen_L; prm.gen_blue = e->gen_blue; prm.chirp = pl->chirp[ps.axis]; prm.bspec = pl->bspec[ps.axis];
        for (int i = 0; i < e->gen_nfac; ++i) prm.gen_fac[i] = e->gen_fac[i];
    }
    // L2 prefetch of the next tile only where the pass's input cannot be sitting in L2 already (measured: a few
    // per cent faster on the 512^3 grids, slightly slower on 256^3 where A1 / A2 are L2 hits anyway)
    {
        const size_t r = pl->d.prec == POISSON_FP64 ? 8 : 4;
        const size_t in_bytes = q == POISSON_PASS_F1 ? (size_t)pl->d.n[0] * pl->d.n[1] * pl->d.n[2] * r
                              : (q == POISSON_PASS_F2 || q == POISSON_PASS_I1) ? (size_t)pl->d.a1_elems * 2 * r
                              : (size_t)pl->a2_alloc_elems * 2 * r;     // chunked: one chunk of A2, written moments ago
        const size_t k_bytes = (size_t)pl->kint_elems * r;
        prm.prefetch = (in_bytes >= pl->pf_min_bytes ? 1 : 0) | (q == POISSON_PASS_F3 && k_bytes >= pl->pf_min_bytes ? 2 : 0);
        if (pl->pf_force[q] >= 0) prm.prefetch = pl->pf_force[q];
    }
    return prm;
}

// The whole solve as one cooperative launch (solve_kernel.cuh).
static int run_fused(poisson_plan *pl, const void *rho, void *V, cudaStream_t st) {
    SolveParams sp;
    for (int q = 0; q < 5; ++q) sp.pass[q] = pass_params(pl, q, rho, V);
    sp.sync = pl->fused_sync;
    sp.n_planes = pl->d.H;
    sp.t2 = pl->tiles_per_g[1]; sp.t3 = pl->tiles_per_g[2];
    sp.skew = pl->fused_skew;
    // the barrier / per-plane counters start from zero on EVERY launch (an aborted launch, or a launch on another
    // stream, must not leave the next one spinning on stale counts)
    PF_CUDA(cudaMemsetAsync(pl->fused_sync, 0, (size_t)(2 + 2 * pl->d.H) * sizeof(unsigned), st));
    void *args[] = {&sp};
    PF_CUDA(cudaLaunchCooperativeKernel(pl->fused->func, dim3(pl->fused_grid), dim3(pl->fused->NT), args,
                                        pl->fused->smem_bytes, st));
    return POISSON_OK;
}

// Launches of one solve in order: F1 | F2, F3, I2 (once, or once per chunk of k_a planes) | I1.
// Chunked plans (large grids): the three middle passes work plane by plane (g = k_a), so they can run chunk by chunk
// through an A2 buffer that holds ONE chunk -- written by F2, transformed in place by F3, consumed by I2 while it is
// still in the 126 MB L2, and overwritten by the next chunk before it is ever evicted: A2's four sweeps (and its
// write-back) stop being HBM traffic (fewer round trips to global memory).
// f(q, prm, grid) -> status, called once per launch; passes outside [first, last] are skipped.
extern "C++" {
template <class F>
static int for_each_launch(const poisson_plan *pl, const void *rho, void *V, const Lane *ln, int first, int last, F &&f) {
    const size_t cplx = 2 * pl->elem_real;
    auto one = [&](int q) -> int { return (q < first || q > last) ? POISSON_OK : f(q, pass_params(pl, q, rho, V, ln), pl->grid[q]); };
    int rc = one(POISSON_PASS_F1);
    if (rc != POISSON_OK) return rc;
    if (pl->n_chunks <= 1) {
        for (int q = POISSON_PASS_F2; q <= POISSON_PASS_I2 && rc == POISSON_OK; ++q) rc = one(q);
    } else {
        const int G = pl->d.H;
        for (int g0 = 0; g0 < G && rc == POISSON_OK; g0 += pl->chunk_planes) {
            const int ng = G - g0 < pl->chunk_planes ? G - g0 : pl->chunk_planes;
            for (int q = POISSON_PASS_F2; q <= POISSON_PASS_I2 && rc == POISSON_OK; ++q) {
                if (q < first || q > last) continue;
                PassParams prm = pass_params(pl, q, rho, V, ln);
                prm.n_tiles = ng * pl->tiles_per_g[q];
                prm.n_tiles1 = prm.n_tiles;
                prm.k_g0 = g0;                                     // K^F is indexed by the plane's position in the whole grid
                if (q == POISSON_PASS_F2) prm.in = static_cast<const char *>(prm.in) + (size_t)g0 * prm.gs_in * cplx;
                if (q == POISSON_PASS_I2) prm.out = static_cast<char *>(prm.out) + (size_t)g0 * prm.gs_out * cplx;
                // the A2 side of the pass addresses the chunk buffer: extents of A2 with chunk_planes along axis a
                {
                    const PlanDesc &d = pl->d;
                    const int a = d.order[0], b = d.order[1], c = d.order[2];
                    long long e[3] = {d.ext2[0], d.ext2[1], d.ext2[2]};
                    e[a] = pl->chunk_planes;
                    auto st = [&](int ax) -> long long { return ax == 0 ? 1 : (ax == 1 ? e[0] : e[0] * e[1]); };
                    const int n_ax = q == POISSON_PASS_F3 ? c : b;                 // transformed axis of this pass
                    const int p_ax = 3 - a - n_ax;                                 // pencil index axis
                    const long long gs = st(a), ns = st(n_ax), ps = st(p_ax);
                    if (q != POISSON_PASS_I2) { prm.gs_out = gs; prm.ns_out = ns; prm.ps_out = ps; }
                    if (q != POISSON_PASS_F2) { prm.gs_in = gs; prm.ns_in = ns; prm.ps_in = ps; }
                }
                rc = f(q, prm, prm.n_tiles < pl->resident[q] ? prm.n_tiles : pl->resident[q]);
            }
        }
    }
    if (rc != POISSON_OK) return rc;
    return one(POISSON_PASS_I1);
}
}  // extern "C++"

// ev: optional, launches_per_solve + 1 events recorded before the first launch and after every launch
static int run_passes(poisson_plan *pl, const void *rho, void *V, cudaStream_t st, int first, int last,
                      cudaEvent_t *ev = nullptr, const Lane *ln = nullptr) {
    if (ev) PF_CUDA(cudaEventRecord(ev[0], st));
    int item = 0;
    return for_each_launch(pl, rho, V, ln, first, last, [&](int q, const PassParams &prm_in, int grid) -> int {
        const KernelEntry *e = pl->k[q];
        PassParams prm = prm_in;
        void *args[] = {&prm};
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(e->NT);
        cfg.dynamicSmemBytes = e->smem_bytes; cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // PDL: prologue overlaps the previous pass's tail
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr; cfg.numAttrs = pl->use_pdl ? 1 : 0;
        PF_CUDA(cudaLaunchKernelExC(&cfg, e->func, args));
        ++item;
        if (ev) PF_CUDA(cudaEventRecord(ev[item], st));
        return POISSON_OK;
    });
}

// Builds the graph of one solve on the plan's own intermediates (explicit kernel nodes, plain dependencies).
// Parameters of pass q restricted to the k_a planes [g0, g0 + ng) (middle passes F2, F3, I2) and / or to the range
// [x0, x0 + nx) (nx = 0: all) of the axis along which F1 / F2 / I2 / I1 do not couple: x when x is processed last (their pencil
// index), else the axis o (b = x: F1 / I1's group index, F2 / I2's pencil index) -- on the full-size arrays.
static PassParams range_params(const poisson_plan *pl, int q, const Lane *ln, int g0, int ng, int x0 = 0, int nx = 0) {
    const size_t cplx = 2 * pl->elem_real;
    PassParams prm = pass_params(pl, q, nullptr, nullptr, ln);
    const bool ends = q == POISSON_PASS_F1 || q == POISSON_PASS_I1;
    long long off_in = 0, off_out = 0;
    if (!ends) {
        prm.k_g0 = g0;                                     // K^F is indexed by the plane's position in the whole grid
        off_in += (long long)g0 * prm.gs_in; off_out += (long long)g0 * prm.gs_out;
    } else {
        ng = (int)pl->d.pass[q].n_g;
    }
    if (nx > 0) {
        const int e = pl->k[q]->P;
        if (ends && pl->d.order[1] == 0) {   // b = x: the range runs along F1 / I1's group index g (the axis o, which is F2 / I2's pencil index)
            ng = nx;
            off_in += (long long)x0 * prm.gs_in; off_out += (long long)x0 * prm.gs_out;
        } else if (ends) {   // c = x: pencils are x-pairs: rho / V in pairs, A1 in complex numbers (two per pair)
            const int x0p = x0 / 2, nxp = nx / 2;
            prm.n_p = nxp; prm.tiles_per_g = (nxp + e - 1) / e;
            if (q == POISSON_PASS_F1) { off_in += (long long)x0p * prm.ps_in; off_out += 2LL * x0p * prm.ps_out; }
            else { off_in += 2LL * x0p * prm.ps_in; off_out += (long long)x0p * prm.ps_out; }
        } else {
            prm.n_p = nx; prm.tiles_per_g = (nx + e - 1) / e;
            off_in += (long long)x0 * prm.ps_in; off_out += (long long)x0 * prm.ps_out;
        }
    }
    prm.n_tiles = ng * prm.tiles_per_g;
    prm.n_tiles1 = prm.n_tiles;
    prm.in = static_cast<const char *>(prm.in) + (size_t)off_in * cplx;
    prm.out = static_cast<char *>(prm.out) + (size_t)off_out * cplx;
    return prm;
}

static int build_graph(poisson_plan *pl, GraphSolve &g, const Lane *ln) {
    if (g.exec) return POISSON_OK;
    PF_CUDA(cudaGraphCreate(&g.graph, 0));
    auto add_node = [&](int q, PassParams prm, int grid, cudaGraphNode_t *node) -> int {
        const KernelEntry *e = pl->k[q];
        void *args[] = {&prm};
        cudaKernelNodeParams kp{};
        kp.func = const_cast<void *>(e->func);
        kp.gridDim = dim3(grid); kp.blockDim = dim3(e->NT);
        kp.sharedMemBytes = (unsigned)e->smem_bytes;
        kp.kernelParams = args; kp.extra = nullptr;
        PF_CUDA(cudaGraphAddKernelNode(node, g.graph, nullptr, 0, &kp));
        return POISSON_OK;
    };
    // data dependency from -> to; programmatic (the dependent may launch when `from` triggers, and waits inside the kernel) when asked
    const bool prog = pl->use_pdl;
    auto add_edge = [&](cudaGraphNode_t from, cudaGraphNode_t to, bool programmatic) -> int {
        if (programmatic) {
            cudaGraphEdgeData ed{};
            ed.type = cudaGraphDependencyTypeProgrammatic; ed.from_port = cudaGraphKernelNodePortProgrammatic;
            PF_CUDA(cudaGraphAddDependencies_v2(g.graph, &from, &to, &ed, 1));
        } else {
            PF_CUDA(cudaGraphAddDependencies(g.graph, &from, &to, 1));
        }
        return POISSON_OK;
    };
    int rc = POISSON_OK;
    const bool shaped = pl->n_chunks <= 1 && !ln;   // batch lanes already overlap each other: plain chains there (measured: 90.3 vs 92.8 us)
    const int B = shaped ? (pl->branches < pl->d.H ? pl->branches : pl->d.H) : 1;
    int R = shaped ? pl->xchains : 1;
    int n_chain = pl->d.n[0];   // points of the chain axis: x when it is processed last, else the axis o (= c when b = x)
    {   // x chains need: no plane chunks, the register engine everywhere, whole tiles per range
        bool ok = R > 1 && pl->n_chunks <= 1;
        for (int q = 0; q < 5 && ok; ++q) ok = !pl->k[q]->generic;
        if (ok && pl->d.order[2] == 0) ok = pl->d.n[0] % (R * 2 * pl->k[0]->P) == 0 && pl->d.n[0] % (R * pl->k[1]->P) == 0;
        else if (ok && pl->d.order[1] == 0) { n_chain = pl->d.n[pl->d.order[2]]; ok = n_chain % (R * pl->k[1]->P) == 0; }
        else ok = false;
        if (!ok) R = 1;
    }
    if (R > 1) {
        // F1_r -> F2_{r,j} -> F3_j -> I2_{r,j} -> I1_r: r = range of x (F1 / F2 / I2 / I1 tiles only couple along y resp. k_a),
        // j = range of k_a planes (F3 couples along x).  Every kernel except F3 has a successor that only needs part of the grid.
        const int J = B > 1 ? B : 1, nxr = n_chain / R;
        std::vector<cudaGraphNode_t> f1(R), i1(R), f2(R * J), f3(J), i2(R * J);
        g.node_f1 = nullptr; g.node_i1 = nullptr;   // rho / V are patched into R nodes each: see run_graph
        g.xr = R;
        for (int r = 0; r < R && rc == POISSON_OK; ++r) {
            g.prm_f1x[r] = range_params(pl, POISSON_PASS_F1, ln, 0, 0, r * nxr, nxr);
            rc = add_node(POISSON_PASS_F1, g.prm_f1x[r], g.prm_f1x[r].n_tiles < pl->grid[0] ? g.prm_f1x[r].n_tiles : pl->grid[0], &f1[r]);
            g.node_f1x[r] = f1[r];
            g.off_rho[r] = (long long)reinterpret_cast<size_t>(g.prm_f1x[r].in);    // built on a NULL rho: the pointer IS the range's offset
        }
        auto pr = [&](int j, int &g0, int &ng) { g0 = (int)((long long)pl->d.H * j / J); ng = (int)((long long)pl->d.H * (j + 1) / J) - g0; };
        for (int q = POISSON_PASS_F2; q <= POISSON_PASS_I2 && rc == POISSON_OK; ++q)
            for (int j = 0; j < J && rc == POISSON_OK; ++j) {
                int g0, ng; pr(j, g0, ng);
                if (q == POISSON_PASS_F3) {
                    const PassParams prm = range_params(pl, q, ln, g0, ng);
                    rc = add_node(q, prm, prm.n_tiles < pl->grid[q] ? prm.n_tiles : pl->grid[q], &f3[j]);
                    for (int r = 0; r < R && rc == POISSON_OK; ++r) rc = add_edge(f2[r * J + j], f3[j], prog && r == 0);
                } else {
                    for (int r = 0; r < R && rc == POISSON_OK; ++r) {
                        const PassParams prm = range_params(pl, q, ln, g0, ng, r * nxr, nxr);
                        cudaGraphNode_t &node = q == POISSON_PASS_F2 ? f2[r * J + j] : i2[r * J + j];
                        rc = add_node(q, prm, prm.n_tiles < pl->grid[q] ? prm.n_tiles : pl->grid[q], &node);
                        if (rc == POISSON_OK) rc = add_edge(q == POISSON_PASS_F2 ? f1[r] : f3[j], node, prog);
                    }
                }
            }
        for (int r = 0; r < R && rc == POISSON_OK; ++r) {
            g.prm_i1x[r] = range_params(pl, POISSON_PASS_I1, ln, 0, 0, r * nxr, nxr);
            rc = add_node(POISSON_PASS_I1, g.prm_i1x[r], g.prm_i1x[r].n_tiles < pl->grid[4] ? g.prm_i1x[r].n_tiles : pl->grid[4], &i1[r]);
            g.node_i1x[r] = i1[r];
            g.off_V[r] = (long long)reinterpret_cast<size_t>(g.prm_i1x[r].out);
            for (int j = 0; j < J && rc == POISSON_OK; ++j) rc = add_edge(i2[r * J + j], i1[r], prog && j == 0);
        }
    } else if (B > 1) {
        // F1 -> B parallel chains (F2 -> F3 -> I2 over a range of k_a planes: the middle passes work plane by plane) -> I1.
        // A chain's next kernel is ready while the other chains still run, so its CTAs fill the slots a draining kernel frees:
        // the ramp-up / tail of the middle passes overlaps other work, as it does between the lanes of a batch.
        g.prm_f1 = pass_params(pl, POISSON_PASS_F1, nullptr, nullptr, ln);
        g.prm_i1 = pass_params(pl, POISSON_PASS_I1, nullptr, nullptr, ln);
        rc = add_node(POISSON_PASS_F1, g.prm_f1, pl->grid[0], &g.node_f1);
        // node creation order matters: chain by chain, I1 last (creating I1 before the chains made the wire grid 50 % slower)
        std::vector<cudaGraphNode_t> tails(B, g.node_f1);
        for (int j = 0; j < B; ++j) {
            const int g0 = (int)((long long)pl->d.H * j / B), g1 = (int)((long long)pl->d.H * (j + 1) / B);
            for (int q = POISSON_PASS_F2; q <= POISSON_PASS_I2 && rc == POISSON_OK; ++q) {
                const PassParams prm = range_params(pl, q, ln, g0, g1 - g0);
                cudaGraphNode_t node;
                rc = add_node(q, prm, prm.n_tiles < pl->grid[q] ? prm.n_tiles : pl->grid[q], &node);
                if (rc == POISSON_OK) rc = add_edge(tails[j], node, prog);
                tails[j] = node;
            }
        }
        if (rc == POISSON_OK) rc = add_node(POISSON_PASS_I1, g.prm_i1, pl->grid[4], &g.node_i1);
        for (size_t j = 0; j < tails.size() && rc == POISSON_OK; ++j) rc = add_edge(tails[j], g.node_i1, prog && j == 0);   // one programmatic edge into I1, the rest plain
    } else {
        cudaGraphNode_t prev = nullptr;
        bool have_prev = false;
        rc = for_each_launch(pl, nullptr, nullptr, ln, 0, 4, [&](int q, const PassParams &prm, int grid) -> int {
            if (q == POISSON_PASS_F1) g.prm_f1 = prm;
            if (q == POISSON_PASS_I1) g.prm_i1 = prm;
            cudaGraphNode_t node;
            int rc1 = add_node(q, prm, grid, &node);
            if (rc1 == POISSON_OK && have_prev) rc1 = add_edge(prev, node, false);
            if (rc1 != POISSON_OK) return rc1;
            if (q == POISSON_PASS_F1) g.node_f1 = node;
            if (q == POISSON_PASS_I1) g.node_i1 = node;
            prev = node; have_prev = true;
            return POISSON_OK;
        });
    }
    if (rc != POISSON_OK) { cudaGraphDestroy(g.graph); g.graph = nullptr; return rc; }
    PF_CUDA(cudaGraphInstantiate(&g.exec, g.graph, 0));
    g.rho = nullptr; g.V = nullptr;
    return POISSON_OK;
}

// The same graph with programmatic-dependent-launch edges: captured from the PDL stream launches (capture turns
// the launch attribute into programmatic edges); the F1 / I1 kernel nodes are identified by their function.
static int build_graph_pdl(poisson_plan *pl, GraphSolve &g, const Lane *ln) {
    if (g.exec) return POISSON_OK;
    if ((pl->branches > 1 || pl->xchains > 1) && pl->n_chunks <= 1 && !ln) {   // parallel chains: explicit nodes with programmatic edges
        const bool saved = pl->use_pdl;
        pl->use_pdl = true;
        const int rc = build_graph(pl, g, ln);
        pl->use_pdl = saved;
        return rc;
    }
    cudaStream_t cs = nullptr;
    PF_CUDA(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    const bool saved = pl->use_pdl;
    pl->use_pdl = true;
    cudaError_t ce = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
    int rc = ce == cudaSuccess ? run_passes(pl, nullptr, nullptr, cs, 0, 4, nullptr, ln) : POISSON_ECUDA;
    cudaGraph_t graph = nullptr;
    if (ce == cudaSuccess) ce = cudaStreamEndCapture(cs, &graph);
    g.prm_f1 = pass_params(pl, POISSON_PASS_F1, nullptr, nullptr, ln);   // as captured (PDL launch order of the prologue)
    g.prm_i1 = pass_params(pl, POISSON_PASS_I1, nullptr, nullptr, ln);
    pl->use_pdl = saved;
    cudaStreamDestroy(cs);
    if (rc != POISSON_OK || ce != cudaSuccess || !graph) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return POISSON_ECUDA; }
    g.graph = graph;
    size_t nn = 0;
    PF_CUDA(cudaGraphGetNodes(graph, nullptr, &nn));
    std::vector<cudaGraphNode_t> nodes(nn);
    PF_CUDA(cudaGraphGetNodes(graph, nodes.data(), &nn));
    int found = 0;
    for (size_t i = 0; i < nn; ++i) {
        cudaGraphNodeType ty;
        if (cudaGraphNodeGetType(nodes[i], &ty) != cudaSuccess || ty != cudaGraphNodeTypeKernel) continue;
        cudaKernelNodeParams kp{};
        PF_CUDA(cudaGraphKernelNodeGetParams(nodes[i], &kp));
        if (kp.func == pl->k[POISSON_PASS_F1]->func) { g.node_f1 = nodes[i]; ++found; }
        if (kp.func == pl->k[POISSON_PASS_I1]->func) { g.node_i1 = nodes[i]; ++found; }
    }
    if (found != 2) { cudaGraphDestroy(g.graph); g.graph = nullptr; g_last_error = "captured graph does not hold the F1 / I1 kernels exactly once"; return POISSON_ECUDA; }
    PF_CUDA(cudaGraphInstantiate(&g.exec, g.graph, 0));
    g.rho = nullptr; g.V = nullptr;
    return POISSON_OK;
}

static int run_graph(poisson_plan *pl, GraphSolve &g, const void *rho, void *V, cudaStream_t st) {
    for (int q = 0; q < 5; q += 4) {
        const bool stale = q == 0 ? g.rho != rho : g.V != V;
        if (!stale) continue;
        const KernelEntry *e = pl->k[q];
        const int parts = g.xr > 1 ? g.xr : 1;
        for (int r = 0; r < parts; ++r) {
            PassParams &prm = g.xr > 1 ? (q == 0 ? g.prm_f1x[r] : g.prm_i1x[r]) : (q == 0 ? g.prm_f1 : g.prm_i1);
            const long long off = g.xr > 1 ? (q == 0 ? g.off_rho[r] : g.off_V[r]) : 0;
            if (q == 0) prm.in = static_cast<const char *>(rho) + off; else prm.out = static_cast<char *>(V) + off;
            void *args[] = {&prm};
            cudaKernelNodeParams kp{};
            kp.func = const_cast<void *>(e->func);
            kp.gridDim = dim3(prm.n_tiles < pl->grid[q] ? prm.n_tiles : pl->grid[q]); kp.blockDim = dim3(e->NT);
            kp.sharedMemBytes = (unsigned)e->smem_bytes;
            kp.kernelParams = args; kp.extra = nullptr;
            const cudaGraphNode_t node = g.xr > 1 ? (q == 0 ? g.node_f1x[r] : g.node_i1x[r]) : (q == 0 ? g.node_f1 : g.node_i1);
            PF_CUDA(cudaGraphExecKernelNodeSetParams(g.exec, node, &kp));   // launch attributes (PDL edges) stay as built
        }
    }
    g.rho = rho; g.V = V;
    PF_CUDA(cudaGraphLaunch(g.exec, st));
    return POISSON_OK;
}

static int run_solve(poisson_plan *pl, const void *rho, void *V, cudaStream_t st) {
    if (pl->fused && pl->use_fused) return run_fused(pl, rho, V, st);
    if (pl->use_graph && active_graph(pl)) {
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) { cudaGetLastError(); cap = cudaStreamCaptureStatusNone; }
        if (cap == cudaStreamCaptureStatusNone) return run_graph(pl, *active_graph(pl), rho, V, st);
        // the caller is capturing `st` into a graph of their own: plain launches become its nodes
    }
    return run_passes(pl, rho, V, st, 0, 4);
}

// Several small solves per launch (poisson_solve_batch on small grids): each of the five launches covers the
// tiles of nbw densities; density bi uses slot bi of the wide intermediates, reads rho[bi] and writes V[bi].
static int run_passes_wide(poisson_plan *pl, const void *const *rho, void *const *V, int nbw, cudaStream_t st) {
    for (int q = 0; q < 5; ++q) {
        const KernelEntry *e = pl->k[q];
        PassParams prm = pass_params(pl, q, nullptr, nullptr);
        prm.n_tiles = nbw * pl->n_tiles[q];
        const long long s1 = pl->d.a1_elems, s2 = pl->d.a2_elems;
        switch (q) {
            case POISSON_PASS_F1: prm.in = nullptr; prm.out = pl->wide_a1; prm.use_list = 1; prm.bs_out = s1; break;
            case POISSON_PASS_F2: prm.in = pl->wide_a1; prm.out = pl->wide_a2; prm.bs_in = s1; prm.bs_out = s2; break;
            case POISSON_PASS_F3: prm.in = pl->wide_a2; prm.out = pl->wide_a2; prm.bs_in = s2; prm.bs_out = s2; break;
            case POISSON_PASS_I2: prm.in = pl->wide_a2; prm.out = pl->wide_a1; prm.bs_in = s2; prm.bs_out = s1; break;
            default: prm.in = pl->wide_a1; prm.out = nullptr; prm.use_list = 2; prm.bs_in = s1; break;
        }
        if (q == POISSON_PASS_F1) for (int i = 0; i < nbw; ++i) prm.blist[i] = rho[i];
        if (q == POISSON_PASS_I1) for (int i = 0; i < nbw; ++i) prm.blist[i] = V[i];
        prm.prefetch = 0;   // the wide intermediates are sized to stay in L2
        void *args[] = {&prm};
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(prm.n_tiles < pl->resident[q] ? prm.n_tiles : pl->resident[q]); cfg.blockDim = dim3(e->NT);
        cfg.dynamicSmemBytes = e->smem_bytes; cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr; cfg.numAttrs = pl->use_pdl ? 1 : 0;
        PF_CUDA(cudaLaunchKernelExC(&cfg, e->func, args));
    }
    return POISSON_OK;
}

// Densities per launch for device batches: small grids only (one density leaves most of the GPU idle: 32^3 -> 64^3
// has 64 .. 264 tiles per pass for 592 resident CTAs), as many as keep the wide intermediates within ~96 MB of L2.
static int wide_width(const poisson_plan *pl, int count) {
    const size_t lane_bytes = (size_t)(pl->d.a1_elems + pl->d.a2_elems) * 2 * pl->elem_real;
    int w = 0;
    if (pl->env_wide >= 0) w = pl->env_wide;
    else if (lane_bytes <= ((size_t)16 << 20)) w = (int)(((size_t)96 << 20) / lane_bytes);   // measured: 64^3 (12.8 MB) gains 18 % over 3 lanes, 96^3 (43 MB) loses
    if (w > PF_MAX_WIDE) w = PF_MAX_WIDE;
    if (w > count) w = count;
    return w >= 2 ? w : 0;
}

// Times the launch modes on scratch inputs (timing does not depend on the values) and keeps the fastest.
static int tune_plan(poisson_plan *pl) {
    const char *e_tune = std::getenv("POISSON_TUNE"), *e_pdl = std::getenv("POISSON_PDL"), *e_fused = std::getenv("POISSON_FUSED");
    const char *e_graph = std::getenv("POISSON_GRAPH");
    if (e_graph && e_graph[0] == '1') {                                                    // forced
        const bool pdl = e_pdl && e_pdl[0] == '1';
        if ((pdl ? build_graph_pdl(pl, pl->gs_pdl, nullptr) : build_graph(pl, pl->gs, nullptr)) == POISSON_OK) pl->use_graph = true; else cudaGetLastError();
        return POISSON_OK;
    }
    if ((e_tune && e_tune[0] == '0') || e_pdl || (e_fused && e_fused[0] == '1')) return POISSON_OK;   // forced / off
    const size_t bytes = (size_t)pl->d.n[0] * pl->d.n[1] * pl->d.n[2] * pl->elem_real;
    // rho / V rotate over a ring whose footprint exceeds the L2 (as a caller's fresh densities do: a ring that stays L2 resident makes
    // F1 look faster than it is and shifts the choice between close candidates); grids whose single density already exceeds half
    // the L2 take one buffer each
    int nring = (int)(((size_t)160 << 20) / (2 * bytes)) + 1;
    if (nring > 8) nring = 8;
    void *ring = nullptr, *rho = nullptr, *V = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaStream_t ts = nullptr;   // a private non-blocking stream: tuning never synchronises with the caller's streams
    int rc = POISSON_OK;
    auto cleanup = [&] { cudaFree(ring); if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); if (ts) cudaStreamDestroy(ts); };
    if (cudaStreamCreateWithFlags(&ts, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return POISSON_OK; }
    const size_t slot = (bytes + 255) & ~(size_t)255;
    if (cudaMalloc(&ring, 2 * slot * nring) != cudaSuccess) {
        cudaGetLastError(); nring = 1;
        if (cudaMalloc(&ring, 2 * slot) != cudaSuccess) { cudaGetLastError(); cleanup(); return POISSON_OK; }   // no room to tune: keep defaults
    }
    rho = ring; V = static_cast<char *>(ring) + slot * nring;
    auto ring_rho = [&](int i) { return static_cast<const void *>(static_cast<const char *>(rho) + slot * (i % nring)); };
    auto ring_V = [&](int i) { return static_cast<void *>(static_cast<char *>(V) + slot * (i % nring)); };
    cudaMemsetAsync(ring, 0, 2 * slot * nring, ts);
    cudaMemsetAsync(pl->kint, 0, (size_t)pl->kint_elems * pl->elem_real, ts);
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { cudaGetLastError(); cleanup(); return POISSON_OK; }
    const bool modes[5][3] = {{false, false, false}, {true, false, false}, {false, true, false}, {false, false, true}, {true, false, true}};   // {pdl, fused, graph}
    int best = 0; float best_ms = 1e30f;
    // ms per solve of the launch mode currently set in the plan (0: failed)
    auto time_mode = [&]() -> float {
        int reps = 3;
        float ms = 0.f, best_round = 1e30f;
        for (int round = 0; round < 3 && rc == POISSON_OK; ++round) {   // round 0: warm-up + pick the repeat count; then the faster of two
            cudaEventRecord(e0, ts);
            for (int i = 0; i < reps && rc == POISSON_OK; ++i) rc = run_solve(pl, ring_rho(i), ring_V(i), ts);
            cudaEventRecord(e1, ts);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = cuda_fail(cudaGetLastError(), "tuning solve"); return 0.f; }
            cudaEventElapsedTime(&ms, e0, e1);
            ms /= (float)reps;
            if (round == 0) { reps = (int)(2.0f / (ms > 1e-4f ? ms : 1e-4f)); reps = reps < 3 ? 3 : (reps > 64 ? 64 : reps); }
            else if (ms < best_round) best_round = ms;
        }
        return best_round;
    };
    // Graph shape: {chains over ranges of k_a planes, chains over ranges of x} (build_graph).  Which shape wins depends on the
    // grid (measured on B200: 128^3 -> 256^3 fp64 98.4 us plain, 92.3 with 4 plane chains, 90.6 with 2 x 2; 32^3 -> 64^3
    // loses 2 us with any), so the shapes are timed like the launch modes; POISSON_BRANCHES / POISSON_XCHAINS fix one.
    static const int shapes[][2] = {{1, 1}, {2, 1}, {4, 1}, {2, 2}, {2, 4}};
    int shape_best[2] = {pl->branches, pl->xchains};
    if (!pl->env_shape && pl->n_chunks <= 1) {
        float sb = 1e30f;
        pl->use_pdl = false; pl->use_fused = false; pl->use_graph = true;
        for (const auto &sh : shapes) {
            if (rc != POISSON_OK) break;
            destroy_graph(pl->gs);
            pl->branches = sh[0]; pl->xchains = sh[1];
            if (build_graph(pl, pl->gs, nullptr) != POISSON_OK) { cudaGetLastError(); g_last_error.clear(); continue; }
            if (sh[1] > 1 && pl->gs.xr <= 1) continue;   // x chains do not apply to this plan: same graph as {sh[0], 1}
            const float ms = time_mode();
            if (rc == POISSON_OK && ms > 0.f && ms < 0.995f * sb) { sb = ms; shape_best[0] = sh[0]; shape_best[1] = sh[1]; }
        }
        destroy_graph(pl->gs);
        pl->branches = shape_best[0]; pl->xchains = shape_best[1];
    }
    if (rc == POISSON_OK && build_graph(pl, pl->gs, nullptr) != POISSON_OK) { cudaGetLastError(); g_last_error.clear(); }      // no graph: that mode is skipped
    if (rc == POISSON_OK && build_graph_pdl(pl, pl->gs_pdl, nullptr) != POISSON_OK) { cudaGetLastError(); g_last_error.clear(); }
    for (int m = 0; m < 5 && rc == POISSON_OK; ++m) {
        if (modes[m][1] && !pl->fused) continue;
        if (modes[m][2] && !(modes[m][0] ? pl->gs_pdl.exec : pl->gs.exec)) continue;
        pl->use_pdl = modes[m][0]; pl->use_fused = modes[m][1]; pl->use_graph = modes[m][2];
        const float ms = time_mode();
        if (rc == POISSON_OK) {
            pl->tune_ms[m] = ms;
            // the timing loop queues launches ahead of the device; a caller that issues one solve at a time pays the host cost of five
            // stream launches (about 4 us each with the call around them) against one graph launch: stream modes count as >= 20 us
            const float eff = (!modes[m][1] && !modes[m][2] && ms < 0.020f) ? 0.020f : ms;
            if (eff < 0.99f * best_ms) { best_ms = eff; best = m; }   // a later mode must win by more than the timing noise
        }
    }
    pl->use_pdl = modes[best][0]; pl->use_fused = modes[best][1]; pl->use_graph = modes[best][2];
    cleanup();
    return rc;
}

int poisson_solve(poisson_plan *pl, const void *rho_dev, void *V_dev, void *stream) {
    if (!pl || !rho_dev || !V_dev) return POISSON_EINVAL;
    if (check_device(pl) != POISSON_OK) return POISSON_EINVAL;
    if (reinterpret_cast<size_t>(rho_dev) % 16 || reinterpret_cast<size_t>(V_dev) % 16) return POISSON_EINVAL;
    if (!pl->kernel_set) return POISSON_ENOKERNEL;
    return run_solve(pl, rho_dev, V_dev, reinterpret_cast<cudaStream_t>(stream));
}

int poisson_solve_profiled(poisson_plan *pl, const void *rho_dev, void *V_dev, void *stream) {
    if (!pl || !rho_dev || !V_dev) return POISSON_EINVAL;
    if (check_device(pl) != POISSON_OK) return POISSON_EINVAL;
    if (reinterpret_cast<size_t>(rho_dev) % 16 || reinterpret_cast<size_t>(V_dev) % 16) return POISSON_EINVAL;
    if (!pl->kernel_set) return POISSON_ENOKERNEL;
    constexpr int kMaxProfiled = 512;
    if (pl->prof_count >= kMaxProfiled) return POISSON_ENOMEM;
    if (!pl->prof_events) pl->prof_events = new (std::nothrow) std::vector<cudaEvent_t>();
    if (!pl->prof_events) return POISSON_ENOMEM;
    const int per = launches_per_solve(pl) + 1;
    while ((int)pl->prof_events->size() < per * (pl->prof_count + 1)) {
        cudaEvent_t e;
        PF_CUDA(cudaEventCreate(&e));
        pl->prof_events->push_back(e);
    }
    cudaEvent_t *ev = pl->prof_events->data() + per * pl->prof_count;
    const int rc = run_passes(pl, rho_dev, V_dev, reinterpret_cast<cudaStream_t>(stream), 0, 4, ev);
    if (rc == POISSON_OK) pl->prof_count++;
    return rc;
}

int poisson_profile_read(poisson_plan *pl, double ms_sum[5], int *n_solves) {
    if (!pl || !ms_sum || !n_solves) return POISSON_EINVAL;
    for (int q = 0; q < 5; ++q) ms_sum[q] = 0.0;
    *n_solves = pl->prof_count;
    const int nl = launches_per_solve(pl), per = nl + 1;
    for (int i = 0; i < pl->prof_count; ++i) {
        cudaEvent_t *ev = pl->prof_events->data() + per * i;
        PF_CUDA(cudaEventSynchronize(ev[nl]));
        for (int item = 0; item < nl; ++item) {   // launch order: F1 | (F2, F3, I2) per chunk | I1
            const int q = item == 0 ? POISSON_PASS_F1 : (item == nl - 1 ? POISSON_PASS_I1 : POISSON_PASS_F2 + (item - 1) % 3);
            float ms = 0.f;
            PF_CUDA(cudaEventElapsedTime(&ms, ev[item], ev[item + 1]));
            ms_sum[q] += (double)ms;
        }
    }
    pl->prof_count = 0;
    return POISSON_OK;
}

int poisson_debug_run_passes(poisson_plan *pl, const void *rho_dev, void *V_dev, void *stream, int first, int last) {
    if (!pl || pl->shard || first < 0 || last > 4 || first > last) return POISSON_EINVAL;
    if (first == 0 && !rho_dev) return POISSON_EINVAL;
    if (last == 4 && !V_dev) return POISSON_EINVAL;
    if (first <= 2 && last >= 2 && !pl->kernel_set) return POISSON_ENOKERNEL;
    if (pl->n_chunks > 1 && !(first == 0 && last == 4)) return POISSON_EUNSUPPORTED;   // A2 holds one chunk at a time
    return run_passes(pl, rho_dev, V_dev, reinterpret_cast<cudaStream_t>(stream), first, last);
}

int poisson_debug_workspace(const poisson_plan *pl, int which, void **ptr, long long dims[3]) {
    if (!pl || pl->shard || !ptr || !dims || (which != 0 && which != 1)) return POISSON_EINVAL;
    if (which == 1 && pl->n_chunks > 1) return POISSON_EUNSUPPORTED;   // chunked plan: A2 is never whole in memory
    const long long *ext = which == 0 ? pl->d.ext1 : pl->d.ext2;
    *ptr = which == 0 ? pl->a1 : pl->a2;
    dims[0] = ext[2]; dims[1] = ext[1]; dims[2] = ext[0];
    return POISSON_OK;
}

// ---- batched solves: several densities, one K^F (the paper's repeated-solve setting)
static int ensure_lanes(poisson_plan *pl, int want, bool staging) {
    if (!pl->lanes) pl->lanes = new (std::nothrow) std::vector<Lane>();
    if (!pl->lanes) return POISSON_ENOMEM;
    if (!pl->fork_ev) PF_CUDA(cudaEventCreateWithFlags(&pl->fork_ev, cudaEventDisableTiming));
    const size_t cplx = 2 * pl->elem_real;
    const size_t bytes = (size_t)pl->d.n[0] * pl->d.n[1] * pl->d.n[2] * pl->elem_real;
    while ((int)pl->lanes->size() < want) {
        Lane ln{};
        const bool first = pl->lanes->empty();
        ln.owns_ws = !first;
        cudaError_t ce = cudaSuccess;
        if (first) { ln.a1 = pl->a1; ln.a2 = pl->a2; }
        else if (pl->test_max_lanes > 0 && (int)pl->lanes->size() >= pl->test_max_lanes) {
            ce = cudaErrorMemoryAllocation;   // injected (tests): exercises the fall-back to the lanes that fit
        } else {
            ce = cudaMalloc(&ln.a1, (size_t)pl->d.a1_elems * cplx);
            if (ce == cudaSuccess) ce = cudaMalloc(&ln.a2, (size_t)pl->a2_alloc_elems * cplx);
            if (ce != cudaSuccess) { cudaFree(ln.a1); ln.a1 = nullptr; ln.a2 = nullptr; ln.owns_ws = false; }
        }
        if (ce == cudaSuccess) ce = cudaStreamCreateWithFlags(&ln.st, cudaStreamNonBlocking);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&ln.done, cudaEventDisableTiming);
        if (ce != cudaSuccess) {
            if (ln.owns_ws && ln.a1) { cudaFree(ln.a1); cudaFree(ln.a2); }
            if (ln.st) cudaStreamDestroy(ln.st);
            if (ln.done) cudaEventDestroy(ln.done);
            cudaGetLastError();
            return ce == cudaErrorMemoryAllocation ? POISSON_ENOMEM : cuda_fail(ce, "batch lane allocation");
        }
        if (ln.owns_ws) pl->workspace_bytes += (size_t)(pl->d.a1_elems + pl->a2_alloc_elems) * cplx;
        pl->lanes->push_back(ln);
    }
    if (staging)
        for (int l = 0; l < want; ++l) {
            Lane &ln = (*pl->lanes)[l];
            if (ln.rho_stage && ln.v_stage) continue;
            cudaError_t ce = ln.rho_stage ? cudaSuccess : cudaMalloc(&ln.rho_stage, bytes);
            if (ce == cudaSuccess) ce = cudaMalloc(&ln.v_stage, bytes);
            if (ce != cudaSuccess) {   // never leave a lane with one staging buffer
                cudaFree(ln.rho_stage); ln.rho_stage = nullptr; ln.v_stage = nullptr;
                cudaGetLastError();
                return ce == cudaErrorMemoryAllocation ? POISSON_ENOMEM : cuda_fail(ce, "batch staging allocation");
            }
        }
    return POISSON_OK;
}

// Lanes of a batch.  Host batches always use 3 (H2D, passes and D2H of neighbouring solves overlap).  Device
// batches use 3 while one lane's intermediates are small enough for several lanes to share the 126 MB L2
// (measured on B200: 128^3 -> 256^3 gains 9 %, 256^3 -> 512^3 with 808 MB per lane loses 4 %), else 1.
static int batch_lanes(const poisson_plan *pl, int count, bool host) {
    const size_t lane_bytes = (size_t)(pl->d.a1_elems + pl->d.a2_elems) * 2 * pl->elem_real;
    // device batches: 2 lanes (with the per-lane solve graphs 128^3 -> 256^3 measures 96.5 / 93.1 / 96.2 / 97.8 us per solve at
    // 1 / 2 / 3 / 4 lanes, the wire grid 51.9 / 55.3 / 58.6 at 2 / 3 / 4: two sets of intermediates still share the L2)
    // (the surface grid, 34 MB per lane, still gains from a third lane: 27.7 vs 30.3 us -- three sets fit the L2)
    int lanes = pl->env_lanes >= 0 ? pl->env_lanes : (host ? 3 : (3 * lane_bytes <= ((size_t)110 << 20) ? 3 : (lane_bytes <= ((size_t)256 << 20) ? 2 : 1)));
    if (lanes < 1) lanes = 1;
    if (lanes > 8) lanes = 8;
    return count < lanes ? count : lanes;
}

static int solve_batch_impl(poisson_plan *pl, const void *const *rho, void *const *V, int count, cudaStream_t user, bool host) {
    if (!pl || !rho || !V || count < 0) return POISSON_EINVAL;
    if (count == 0) return POISSON_OK;
    for (int i = 0; i < count; ++i) {
        if (!rho[i] || !V[i]) return POISSON_EINVAL;
        if (!host && (reinterpret_cast<size_t>(rho[i]) % 16 || reinterpret_cast<size_t>(V[i]) % 16)) return POISSON_EINVAL;
    }
    if (!pl->kernel_set) return POISSON_ENOKERNEL;
    if (check_device(pl) != POISSON_OK) return POISSON_EINVAL;
    if (!host) {
        const int W = wide_width(pl, count);
        if (W) {
            if (pl->wide_w < W) {   // allocated once, for the widest launch this grid will ever take
                const int cap = wide_width(pl, PF_MAX_WIDE) > W ? wide_width(pl, PF_MAX_WIDE) : W;
                cudaFree(pl->wide_a1); cudaFree(pl->wide_a2); pl->wide_a1 = pl->wide_a2 = nullptr;
                if (pl->wide_w) pl->workspace_bytes -= (size_t)pl->wide_w * (pl->d.a1_elems + pl->d.a2_elems) * 2 * pl->elem_real;
                pl->wide_w = 0;
                cudaError_t ce = cudaMalloc(&pl->wide_a1, (size_t)cap * pl->d.a1_elems * 2 * pl->elem_real);
                if (ce == cudaSuccess) ce = cudaMalloc(&pl->wide_a2, (size_t)cap * pl->d.a2_elems * 2 * pl->elem_real);
                if (ce != cudaSuccess) { cudaGetLastError(); return ce == cudaErrorMemoryAllocation ? POISSON_ENOMEM : cuda_fail(ce, "wide batch allocation"); }
                pl->wide_w = cap;
                pl->workspace_bytes += (size_t)cap * (pl->d.a1_elems + pl->d.a2_elems) * 2 * pl->elem_real;
            }
            for (int i = 0; i < count; i += W) {
                const int rc1 = run_passes_wide(pl, rho + i, V + i, count - i < W ? count - i : W, user);
                if (rc1 != POISSON_OK) return rc1;
            }
            return POISSON_OK;
        }
    }
    const int L = batch_lanes(pl, count, host);
    if (L == 1 && !host) {   // one lane: the plan's own intermediates on the caller's stream, in the plan's tuned launch mode
        for (int i = 0; i < count; ++i) {
            const int rc1 = run_solve(pl, rho[i], V[i], user);
            if (rc1 != POISSON_OK) return rc1;
        }
        return POISSON_OK;
    }
    int L_use = L;
    int rc = ensure_lanes(pl, L_use, host);
    while (rc == POISSON_ENOMEM && L_use > 1) rc = ensure_lanes(pl, --L_use, host);   // no room for every lane: use the ones that fit
    if (rc != POISSON_OK) return rc;
    const size_t bytes = (size_t)pl->d.n[0] * pl->d.n[1] * pl->d.n[2] * pl->elem_real;
    PF_CUDA(cudaEventRecord(pl->fork_ev, user));                      // the lanes start after the caller's earlier work
    for (int l = 0; l < L_use; ++l) PF_CUDA(cudaStreamWaitEvent((*pl->lanes)[l].st, pl->fork_ev, 0));
    const bool lane_graphs = pl->use_graph && active_graph(pl) && pl->env_lane_graph;
    // one solve on its lane; any failure falls through to the join below so that the caller's stream stays ordered
    // after the lane work already queued
    auto queue_one = [&](int i) -> int {
        Lane &ln = (*pl->lanes)[i % L_use];
        const void *r = rho[i];
        void *v = V[i];
        if (host) {
            PF_CUDA(cudaMemcpyAsync(ln.rho_stage, rho[i], bytes, cudaMemcpyHostToDevice, ln.st));
            r = ln.rho_stage; v = ln.v_stage;
        }
        int rc1;
        if (lane_graphs) {
            if (!ln.gs) {
                ln.gs = new (std::nothrow) GraphSolve();
                if (!ln.gs) return POISSON_ENOMEM;
                std::memset(ln.gs, 0, sizeof(GraphSolve));
            }
            if (!ln.gs->exec) {   // first use, or a kernel switch (set_kernel_even / _complex / back) dropped the lane's graph
                rc1 = pl->use_pdl ? build_graph_pdl(pl, *ln.gs, &ln) : build_graph(pl, *ln.gs, &ln);
                if (rc1 != POISSON_OK) return rc1;
            }
            rc1 = run_graph(pl, *ln.gs, r, v, ln.st);
        } else {
            rc1 = run_passes(pl, r, v, ln.st, 0, 4, nullptr, &ln);
        }
        if (rc1 != POISSON_OK) return rc1;
        if (host) PF_CUDA(cudaMemcpyAsync(V[i], ln.v_stage, bytes, cudaMemcpyDeviceToHost, ln.st));
        return POISSON_OK;
    };
    for (int i = 0; i < count && rc == POISSON_OK; ++i) rc = queue_one(i);
    for (int l = 0; l < L_use; ++l) {                                  // join: the caller's stream continues after every lane
        cudaError_t ce = cudaEventRecord((*pl->lanes)[l].done, (*pl->lanes)[l].st);
        if (ce == cudaSuccess) ce = cudaStreamWaitEvent(user, (*pl->lanes)[l].done, 0);
        if (ce != cudaSuccess && rc == POISSON_OK) rc = cuda_fail(ce, "batch join");
    }
    if (host) { const cudaError_t ce = cudaStreamSynchronize(user); if (ce != cudaSuccess && rc == POISSON_OK) rc = cuda_fail(ce, "batch sync"); }
    return rc;
}

int poisson_plan_batch_lanes(const poisson_plan *pl, int count, int host) {
    return pl && count > 0 ? batch_lanes(pl, count, host != 0) : 0;
}

int poisson_plan_batch_width(const poisson_plan *pl, int count) {
    return pl && count > 0 ? wide_width(pl, count) : 0;
}

int poisson_solve_batch(poisson_plan *pl, const void *const *rho_dev, void *const *V_dev, int count, void *stream) {
    return solve_batch_impl(pl, rho_dev, V_dev, count, reinterpret_cast<cudaStream_t>(stream), false);
}

int poisson_solve_batch_host(poisson_plan *pl, const void *const *rho_host, void *const *V_host, int count, void *stream) {
    return solve_batch_impl(pl, rho_host, V_host, count, reinterpret_cast<cudaStream_t>(stream), true);
}

int poisson_solve_host(poisson_plan *pl, const void *rho_host, void *V_host, void *stream) {
    if (!pl || !rho_host || !V_host) return POISSON_EINVAL;
    if (check_device(pl) != POISSON_OK) return POISSON_EINVAL;
    if (!pl->kernel_set) return POISSON_ENOKERNEL;
    const size_t bytes = (size_t)pl->d.n[0] * pl->d.n[1] * pl->d.n[2] * pl->elem_real;
    if (!pl->rho_stage) {
        cudaError_t ce = cudaMalloc(&pl->rho_stage, bytes);
        if (ce == cudaSuccess) ce = cudaMalloc(&pl->v_stage, bytes);
        if (ce != cudaSuccess) { cudaGetLastError(); return ce == cudaErrorMemoryAllocation ? POISSON_ENOMEM : cuda_fail(ce, "staging allocation"); }
    }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    PF_CUDA(cudaMemcpyAsync(pl->rho_stage, rho_host, bytes, cudaMemcpyHostToDevice, st));
    const int rc = run_solve(pl, pl->rho_stage, pl->v_stage, st);
    if (rc != POISSON_OK) return rc;
    PF_CUDA(cudaMemcpyAsync(V_host, pl->v_stage, bytes, cudaMemcpyDeviceToHost, st));
    PF_CUDA(cudaStreamSynchronize(st));
    return POISSON_OK;
}

// ------------------------------------------------------------------ one solve sharded over several GPUs
static void fill_shard_info(const PlanDesc &d, const ShardDesc &sh, poisson_shard_info *I) {
    std::memset(I, 0, sizeof(*I));
    const long long cplx = d.prec == POISSON_FP64 ? 16 : 8;
    I->rank = sh.rank; I->nranks = sh.R; I->split_axis = sh.o; I->plane_axis = sh.a;
    I->o0 = sh.o0; I->o1 = sh.o1; I->k0 = sh.k0; I->k1 = sh.k1;
    for (int q = 0; q < 3; ++q) { I->local_dims[q] = sh.ext_rho[2 - q]; I->mid_dims[q] = sh.ext_mid[2 - q]; I->back_dims[q] = sh.ext_back[2 - q]; }
    I->mid_bytes = sh.mid_elems * cplx; I->back_bytes = sh.back_elems * cplx;
    // exchange 1: this rank's F1 output (H planes x its o slab x N_x) minus the planes it owns itself;
    // exchange 2: its I2 output (its planes x all o x N_x) minus its own o slab
    const long long no = sh.o1 - sh.o0, ng = sh.k1 - sh.k0, nx = d.ext1[0];
    I->sent_bytes[0] = (d.H - ng) * no * nx * cplx;
    I->sent_bytes[1] = ng * (d.n[sh.o] - no) * nx * cplx;
}

int poisson_shard_describe(int nx, int ny, int nz, const int bc[3], int precision, int rank, int nranks, poisson_shard_info *info) {
    if (!info) return POISSON_EINVAL;
    PlanDesc d;
    int st = plan_build(nx, ny, nz, bc, precision, d);
    if (st != POISSON_OK) return st;
    ShardDesc sh;
    st = shard_build(d, rank, nranks, sh);
    if (st != POISSON_OK) return st;
    static const int kinds[5] = {KIND_F1S, KIND_F2, KIND_F3, KIND_I2S, KIND_I1};
    for (int q = 0; q < 5; ++q)
        if (!find_kernel(kinds[q], sh.pass[q].S, sh.pass[q].pruned, sh.pass[q].lanes_p, precision, 0)) return POISSON_EUNSUPPORTED;
    fill_shard_info(d, sh, info);
    return POISSON_OK;
}

int poisson_shard_plan_create(poisson_plan **out, int nx, int ny, int nz, const int bc[3], double h, int precision, int rank, int nranks) {
    if (!out) return POISSON_EINVAL;
    *out = nullptr;
    if (!(h > 0.0) || !std::isfinite(h)) return POISSON_EINVAL;
    PlanDesc d;
    int st = plan_build(nx, ny, nz, bc, precision, d);
    if (st != POISSON_OK) return st;
    ShardDesc sh;
    st = shard_build(d, rank, nranks, sh);
    if (st != POISSON_OK) return st;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); g_last_error = "no CUDA device"; return POISSON_EARCH; }
    int dev = 0;
    PF_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    PF_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) { g_last_error = "device is sm_" + std::to_string(prop.major * 10 + prop.minor) + ", kernels are sm_100a"; return POISSON_EARCH; }
    poisson_plan *pl = new (std::nothrow) poisson_plan();
    if (!pl) return POISSON_ENOMEM;
    std::memset(static_cast<void *>(pl), 0, sizeof(*pl));
    pl->shard = new (std::nothrow) ShardDesc(sh);
    if (!pl->shard) { delete pl; return POISSON_ENOMEM; }
    pl->d = d; pl->h = h; pl->device = dev; pl->num_sms = prop.multiProcessorCount;
    pl->elem_real = precision == POISSON_FP64 ? 8 : 4;
    pl->late_tw = 1; pl->pdl_trigger = 1; pl->branches = 1; pl->xchains = 1; pl->n_chunks = 1; pl->chunk_planes = d.H;
    pl->env_lanes = pl->env_wide = -1;
    for (int q = 0; q < 5; ++q) pl->pf_force[q] = -1;
    pl->pf_min_bytes = (size_t)96 << 20;
    static const int kinds[5] = {KIND_F1S, KIND_F2, KIND_F3, KIND_I2S, KIND_I1};
    for (int q = 0; q < 5; ++q) {
        const PassDesc &ps = sh.pass[q];
        const KernelEntry *e = find_kernel(kinds[q], ps.S, ps.pruned, ps.lanes_p, precision, 0);
        if (!e) { free_plan(pl); return POISSON_EUNSUPPORTED; }
        pl->k[q] = e;
        pl->tiles_per_g[q] = (int)((ps.n_p + e->P - 1) / e->P);
        pl->n_tiles[q] = (int)(ps.n_g * pl->tiles_per_g[q]);
        cudaError_t ce = cudaFuncSetAttribute(e->func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)e->smem_bytes);
        int occ = 0;
        if (ce == cudaSuccess) ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, e->func, e->NT, e->smem_bytes);
        if (ce != cudaSuccess || occ < 1) { free_plan(pl); return cuda_fail(ce, "shard kernel setup"); }
        pl->resident[q] = occ * pl->num_sms;
        pl->grid[q] = pl->n_tiles[q] < pl->resident[q] ? pl->n_tiles[q] : pl->resident[q];
    }
    const size_t cplx = 2 * pl->elem_real;
    pl->a2_alloc_elems = sh.a2_elems;
    pl->kint_elems = kint_reals(pl);
    size_t ws = 0;
    cudaError_t ce = cudaMalloc(&pl->a2, (size_t)sh.a2_elems * cplx); ws += (size_t)sh.a2_elems * cplx;
    if (ce == cudaSuccess) { ce = cudaMalloc(&pl->kint, (size_t)pl->kint_elems * pl->elem_real); ws += (size_t)pl->kint_elems * pl->elem_real; }
    for (int q = 0; q < 3 && ce == cudaSuccess; ++q) {
        std::vector<unsigned char> host;
        fill_twiddles(host, d.s[q], precision);
        ce = cudaMalloc(&pl->tw[q], host.size());
        if (ce == cudaSuccess) ce = cudaMemcpy(pl->tw[q], host.data(), host.size(), cudaMemcpyHostToDevice);
        ws += host.size();
    }
    if (ce != cudaSuccess) {
        free_plan(pl);
        if (ce == cudaErrorMemoryAllocation) { cudaGetLastError(); return POISSON_ENOMEM; }
        return cuda_fail(ce, "shard workspace allocation");
    }
    pl->workspace_bytes = ws;
    pl->d.info.workspace_bytes = (long long)ws;
    *out = pl;
    return POISSON_OK;
}

int poisson_shard_get_info(const poisson_plan *pl, poisson_shard_info *info) {
    if (!pl || !pl->shard || !info) return POISSON_EINVAL;
    fill_shard_info(pl->d, *pl->shard, info);
    info->workspace_bytes = (long long)pl->workspace_bytes;
    return POISSON_OK;
}

int poisson_shard_set_slabs(poisson_plan *pl, void *const *mid_of_rank, void *const *back_of_rank) {
    if (!pl || !pl->shard || !mid_of_rank || !back_of_rank) return POISSON_EINVAL;
    if (check_device(pl, true) != POISSON_OK) return POISSON_EINVAL;   // the pointers must be valid on the plan's device
    for (int s = 0; s < pl->shard->R; ++s) {
        if (!mid_of_rank[s] || !back_of_rank[s]) return POISSON_EINVAL;
        if (reinterpret_cast<size_t>(mid_of_rank[s]) % 32 || reinterpret_cast<size_t>(back_of_rank[s]) % 32) return POISSON_EINVAL;   // 256-bit pair stores
        pl->sh_mid[s] = mid_of_rank[s]; pl->sh_back[s] = back_of_rank[s];
    }
    pl->sh_slabs_set = true;
    return POISSON_OK;
}

int poisson_shard_set_kernel(poisson_plan *pl, const void *K_f_dev, void *stream) {
    if (!pl || !K_f_dev) return POISSON_EINVAL;
    if (reinterpret_cast<size_t>(K_f_dev) % 16) return POISSON_EINVAL;
    if (check_device(pl, true) != POISSON_OK) return POISSON_EINVAL;
    const int rc = relayout_kernel_spectrum(pl, K_f_dev, false, reinterpret_cast<cudaStream_t>(stream));
    if (rc != POISSON_OK) return rc;
    pl->kernel_set = true;
    return POISSON_OK;
}

// Parameters of pass q of a shard plan on the rank's local arrays.
static PassParams shard_pass_params(const poisson_plan *pl, int q, const void *rho, void *V) {
    const ShardDesc &sh = *pl->shard;
    const PlanDesc &d = pl->d;
    const PassDesc &ps = sh.pass[q];
    PassParams prm{};
    void *mid = pl->sh_mid[sh.rank], *back = pl->sh_back[sh.rank];
    switch (q) {
        case POISSON_PASS_F1: prm.in = rho; prm.out = nullptr; break;
        case POISSON_PASS_F2: prm.in = mid; prm.out = pl->a2; break;
        case POISSON_PASS_F3: prm.in = pl->a2; prm.out = pl->a2; break;
        case POISSON_PASS_I2: prm.in = pl->a2; prm.out = nullptr; break;
        default: prm.in = back; prm.out = V; break;
    }
    prm.kint = pl->kint;
    prm.tw = pl->tw[ps.axis];
    prm.gs_in = ps.gs_in; prm.ns_in = ps.ns_in; prm.ps_in = ps.ps_in;
    prm.gs_out = ps.gs_out; prm.ns_out = ps.ns_out; prm.ps_out = ps.ps_out;
    prm.n_p = (int)ps.n_p; prm.tiles_per_g = pl->tiles_per_g[q]; prm.n_tiles = pl->n_tiles[q]; prm.n_tiles1 = pl->n_tiles[q];
    prm.late_tw = 1; prm.pdl_trigger = 1;
    prm.prefetch = q == POISSON_PASS_F3 && (size_t)pl->kint_elems * pl->elem_real >= pl->pf_min_bytes ? 2 : 0;
    if (q == POISSON_PASS_F1 || q == POISSON_PASS_I2) {
        const bool f1 = q == POISSON_PASS_F1;
        const int T = f1 ? d.H : d.n[sh.o];                 // the distributed axis of the output: k_a planes resp. the split axis o
        prm.sh_R = sh.R; prm.sh_total = T;
        prm.sh_vslow = f1 ? (sh.a > sh.o) : (sh.o > sh.a);
        prm.sh_nx = (int)d.ext1[0];
        prm.sh_eu = f1 ? d.n[sh.o] : d.H;                    // whole extent of the other axis
        prm.sh_u0 = f1 ? sh.o0 : sh.k0;
        prm.sh_vp = (!f1 && d.order[1] == 0) ? 1 : 0;        // I2 along x: the split coordinate is the pencil index
        for (int s = 0; s <= sh.R; ++s) prm.sh_lo[s] = shard_lo(T, s, sh.R);
        for (int s = 0; s < sh.R; ++s) prm.blist[s] = f1 ? pl->sh_mid[s] : pl->sh_back[s];
    }
    return prm;
}

static int shard_launch(poisson_plan *pl, int q, const void *rho, void *V, cudaStream_t st) {
    const KernelEntry *e = pl->k[q];
    PassParams prm = shard_pass_params(pl, q, rho, V);
    void *args[] = {&prm};
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(pl->grid[q]); cfg.blockDim = dim3(e->NT);
    cfg.dynamicSmemBytes = e->smem_bytes; cfg.stream = st;
    PF_CUDA(cudaLaunchKernelExC(&cfg, e->func, args));
    return POISSON_OK;
}

static int shard_ready(const poisson_plan *pl) {
    if (!pl) return POISSON_EINVAL;
    if (check_device(pl, true) != POISSON_OK) return POISSON_EINVAL;
    if (!pl->sh_slabs_set) { g_last_error = "poisson_shard_set_slabs has not been called"; return POISSON_EINVAL; }
    return POISSON_OK;
}

int poisson_shard_forward(poisson_plan *pl, const void *rho_local_dev, void *stream) {
    if (!rho_local_dev || reinterpret_cast<size_t>(rho_local_dev) % 16) return POISSON_EINVAL;
    const int rc = shard_ready(pl);
    if (rc != POISSON_OK) return rc;
    return shard_launch(pl, POISSON_PASS_F1, rho_local_dev, nullptr, reinterpret_cast<cudaStream_t>(stream));
}

int poisson_shard_middle(poisson_plan *pl, void *stream) {
    int rc = shard_ready(pl);
    if (rc != POISSON_OK) return rc;
    if (!pl->kernel_set) return POISSON_ENOKERNEL;
    for (int q = POISSON_PASS_F2; q <= POISSON_PASS_I2 && rc == POISSON_OK; ++q)
        rc = shard_launch(pl, q, nullptr, nullptr, reinterpret_cast<cudaStream_t>(stream));
    return rc;
}

int poisson_shard_inverse(poisson_plan *pl, void *V_local_dev, void *stream) {
    if (!V_local_dev || reinterpret_cast<size_t>(V_local_dev) % 16) return POISSON_EINVAL;
    const int rc = shard_ready(pl);
    if (rc != POISSON_OK) return rc;
    return shard_launch(pl, POISSON_PASS_I1, nullptr, V_local_dev, reinterpret_cast<cudaStream_t>(stream));
}

// ---------------------------------------------------------------------------------------------------------------------
// poisson_solve_static: one whole solve that allocates NO device memory (include/poisson.h has the user-facing text).
//
// The five passes are the same kernels poisson_solve launches; what differs is where their scratch lives.  A plan keeps
// the intermediates A1 / A2, the re-laid K^F copy and the twiddle tables in buffers it cudaMalloc'ed.  Here all of them
// sit in ONE file-scope device array that is part of the library image, so a process that may not (or cannot) allocate
// device memory -- its HBM is already handed out to its own pool, or an allocation failure / the implicit device
// synchronisation of cudaMalloc / cudaFree is not acceptable where the call sits -- can still solve a small grid.
// Price: every device that loads this library holds POISSON_STATIC_SCRATCH_BYTES until the process exits.
//
// Host code must not pass `pf_static_scratch` itself to a kernel: in host code that name is the host-side shadow of
// the symbol, not a device address.  The device address is asked for once per device (static_device_state below) with
// cudaGetSymbolAddress while that device is current, and only that pointer is handed to the kernels.
static __device__ __align__(256) unsigned char pf_static_scratch[POISSON_STATIC_SCRATCH_BYTES];

namespace {

constexpr size_t PF_STATIC_SLOT = (size_t)PF_GENERIC_MAX_S * 16;   // one table of the longest length, fp64 complex
constexpr size_t PF_STATIC_TABLES = 9 * PF_STATIC_SLOT;            // per axis: twiddles, Bluestein chirp, Bluestein spectrum
constexpr int PF_STATIC_MAX_DEV = 64;

struct StaticDeviceState {
    bool ready;               // cudaGetSymbolAddress done for this device
    unsigned char *base;      // device address of pf_static_scratch ON THIS DEVICE
    int num_sms;
    int tab_S[3], tab_L[3], tab_prec[3];   // what the three table slots of this device's array hold right now (0 = nothing)
    poisson_plan *pl;         // host-side description of the last grid solved here; owns NO device memory (never free_plan it)
};
StaticDeviceState g_static_dev[PF_STATIC_MAX_DEV];
std::mutex g_static_mutex;

inline size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

}  // namespace

// First call on a device: checks the architecture and resolves the array's device address.  No allocation.
static int static_device_state(StaticDeviceState **out) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); g_last_error = "no CUDA device"; return POISSON_EARCH; }
    int dev = 0;
    PF_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= PF_STATIC_MAX_DEV) { g_last_error = "device ordinal above 63"; return POISSON_EUNSUPPORTED; }
    StaticDeviceState &sd = g_static_dev[dev];
    if (!sd.ready) {
        int major = 0, sms = 0;
        PF_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        PF_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        if (major != 10) { g_last_error = "device is not compute capability 10.x, kernels are sm_100a"; return POISSON_EARCH; }
        void *ptr = nullptr;
        const cudaError_t ce = cudaGetSymbolAddress(&ptr, pf_static_scratch);   // the address on the CURRENT device
        if (ce != cudaSuccess || !ptr) return cuda_fail(ce, "cudaGetSymbolAddress(pf_static_scratch)");
        sd.base = static_cast<unsigned char *>(ptr);
        sd.num_sms = sms;
        sd.ready = true;
    }
    *out = &sd;
    return POISSON_OK;
}

int poisson_solve_static(int nx, int ny, int nz, const int bc[3], int precision, const void *K_f_dev, const void *rho_dev,
                         void *V_dev, void *stream) {
    if (!bc || !K_f_dev || !rho_dev || !V_dev) return POISSON_EINVAL;
    if (reinterpret_cast<size_t>(K_f_dev) % 16 || reinterpret_cast<size_t>(rho_dev) % 16 || reinterpret_cast<size_t>(V_dev) % 16) return POISSON_EINVAL;
    PlanDesc d;
    int st = plan_build(nx, ny, nz, bc, precision, d);
    if (st != POISSON_OK) return st;
    cudaStream_t cs = reinterpret_cast<cudaStream_t>(stream);

    std::lock_guard<std::mutex> guard(g_static_mutex);   // the host-side records below are shared by every caller
    StaticDeviceState *sd = nullptr;
    st = static_device_state(&sd);
    if (st != POISSON_OK) return st;

    // host-side description of the grid (kernels, tiles, grids): rebuilt only when the grid differs from the last call's
    poisson_plan *pl = sd->pl;
    const bool same = pl && pl->d.prec == precision && !std::memcmp(pl->d.n, d.n, sizeof(d.n)) && !std::memcmp(pl->d.bc, d.bc, sizeof(d.bc));
    if (!same) {
        delete pl;             // plain delete: its pointers are offsets into the static array, there is nothing to cudaFree
        sd->pl = nullptr;
        pl = new (std::nothrow) poisson_plan();
        if (!pl) return POISSON_ENOMEM;
        std::memset(static_cast<void *>(pl), 0, sizeof(*pl));
        int dev = 0;
        cudaGetDevice(&dev);
        pl->d = d; pl->h = 1.0; pl->device = dev; pl->num_sms = sd->num_sms;
        pl->elem_real = precision == POISSON_FP64 ? 8 : 4;
        pl->late_tw = 1; pl->pdl_trigger = 1; pl->branches = 1; pl->xchains = 1; pl->env_lanes = -1; pl->env_wide = -1;
        pl->pf_min_bytes = (size_t)96 << 20;
        for (int q = 0; q < 5; ++q) pl->pf_force[q] = -1;
        for (int q = 0; q < 5; ++q) {
            st = setup_pass(pl, q, false);                 // same kernel choice as poisson_plan_create
            if (st != POISSON_OK) { delete pl; return st; }
        }
        pl->chunk_planes = d.H; pl->n_chunks = 1; pl->a2_alloc_elems = d.a2_elems;
        pl->kint_elems = kint_reals(pl);
        // carve the array: [tables | A1 | A2 | K^F copy], 256-byte aligned pieces
        const size_t cplx = 2 * pl->elem_real;
        const size_t o_a1 = PF_STATIC_TABLES;
        const size_t o_a2 = o_a1 + align256((size_t)d.a1_elems * cplx);
        const size_t o_k = o_a2 + align256((size_t)d.a2_elems * cplx);
        const size_t need = o_k + align256((size_t)pl->kint_elems * pl->elem_real);
        if (need > (size_t)POISSON_STATIC_SCRATCH_BYTES) {
            g_last_error = "poisson_solve_static: this grid needs " + std::to_string(need) + " bytes of scratch, the static array holds " +
                           std::to_string((size_t)POISSON_STATIC_SCRATCH_BYTES) + " (use a plan: poisson_plan_create / poisson_solve)";
            delete pl;
            return POISSON_EUNSUPPORTED;
        }
        pl->a1 = sd->base + o_a1; pl->a2 = sd->base + o_a2; pl->kint = sd->base + o_k;
        for (int q = 0; q < 3; ++q) {
            pl->tw[q] = sd->base + (size_t)(3 * q) * PF_STATIC_SLOT;
            pl->chirp[q] = sd->base + (size_t)(3 * q + 1) * PF_STATIC_SLOT;
            pl->bspec[q] = sd->base + (size_t)(3 * q + 2) * PF_STATIC_SLOT;
        }
        pl->workspace_bytes = need;
        pl->d.info.workspace_bytes = (long long)need;
        sd->pl = pl;
    }

    // twiddle tables: the array keeps the last call's, so an axis is uploaded only when its length or precision changed.
    // Stream-ordered on the caller's stream, in front of the passes that read them.
    for (int q = 0; q < 3; ++q) {
        int M = 0;
        for (int ps = 0; ps < 5; ++ps) if (d.pass[ps].axis == q && pl->k[ps]->generic && pl->k[ps]->gen_blue) M = pl->k[ps]->gen_L;
        const int L = M ? M : d.s[q];
        if (sd->tab_S[q] == d.s[q] && sd->tab_L[q] == L && sd->tab_prec[q] == precision + 1) continue;
        sd->tab_S[q] = 0;                                   // not valid while the upload may fail half way
        std::vector<unsigned char> host;
        fill_twiddles(host, L, precision);
        PF_CUDA(cudaMemcpyAsync(pl->tw[q], host.data(), host.size(), cudaMemcpyHostToDevice, cs));
        if (M) {
            std::vector<unsigned char> hc, hb;
            fill_bluestein(hc, hb, d.s[q], M, precision);
            PF_CUDA(cudaMemcpyAsync(pl->chirp[q], hc.data(), hc.size(), cudaMemcpyHostToDevice, cs));
            PF_CUDA(cudaMemcpyAsync(pl->bspec[q], hb.data(), hb.size(), cudaMemcpyHostToDevice, cs));
        }
        // pageable source: the runtime has staged the bytes when cudaMemcpyAsync returns, the vectors may go
        sd->tab_S[q] = d.s[q]; sd->tab_L[q] = L; sd->tab_prec[q] = precision + 1;
    }

    // K^F of THIS call into the order pass F3 streams it in (nothing of an earlier call's copy is reused: the caller may
    // have changed the kernel), then the five passes.  Every byte of A1 / A2 / the K^F copy that a pass reads was written
    // earlier in this same call, so nothing in the array has to be cleared between calls.
    st = relayout_kernel_spectrum(pl, K_f_dev, false, cs);
    if (st != POISSON_OK) return st;
    return run_passes(pl, rho_dev, V_dev, cs, 0, 4);
}

}  // extern "C"
