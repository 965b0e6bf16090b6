/*
 * poisson.h -- C ABI of the B200-native (sm_100a) Fourier-space Poisson solve of arxiv 1211.5244
 * (Dugan, Genovese, Goedecker, "A Customized 3D GPU Poisson Solver for Free Boundary Conditions").
 *
 * The library computes, for a real density rho on an nx*ny*nz grid,
 *
 *      V = IDFT3( K^F . DFT3( pad(rho) ) ) restricted to the physical box          (Eq. 3)
 *
 * on a grid zero-padded to S_i = 2 N_i along every free axis and S_i = N_i along every periodic
 * axis, which equals the discrete convolution of Eq. 2
 *
 *      V[i] = sum_{i' in box} K[(i - i') mod S] rho[i'],   i in box.
 *
 * The transform is the paper's "customized 3D FFT": zero-padded regions are
 * never read or transformed, the first processed axis is real-to-complex, the K^F multiply is
 * fused between the last forward and first inverse 1D transforms, and only the physical
 * octant / quarter / half is written back.  Every step runs in hand-written CUDA kernels;
 * there is no cuFFT, no CPU fallback, and every entry point fails with a status code (never
 * aborts, never throws) when it cannot run.
 *
 * Conventions (readings of the paper, DESIGN.md section "Readings"):
 *   - arrays are dense C order [z][y][x], x fastest;
 *   - data sits in the first half [0,N) of a padded axis, zeros in [N,2N)   (reading 1);
 *   - forward DFT sign exp(-2 pi i jk/S); forward and inverse are unnormalised and the library
 *     applies 1/(S_x S_y S_z) itself (reading 2); no h^3 volume element is applied (reading 3).
 *
 * Pointer kinds are stated per argument: "device" = CUDA device memory on the current device,
 * "host" = ordinary or pinned host memory.  `stream` is a cudaStream_t passed as void*
 * (NULL = the legacy default stream).
 */
#ifndef POISSON_B200_H
#define POISSON_B200_H

#include <stddef.h>

#if defined(__GNUC__)
#define POISSON_API __attribute__((visibility("default")))
#else
#define POISSON_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct poisson_plan poisson_plan; /* opaque; owned by the library */

enum { POISSON_BC_FREE = 0, POISSON_BC_PERIODIC = 1 };          /* B_i = 2 / 1 of PAPER.md:51 */
enum { POISSON_FP64 = 0, POISSON_FP32 = 1 };
enum {
    POISSON_OK = 0,
    POISSON_EINVAL = 1,       /* null pointer, n <= 0, bc / precision out of range, bad h, misaligned pointer */
    POISSON_EUNSUPPORTED = 2, /* a padded length S_i above the any-length kernel's limit (4096)        */
    POISSON_ENOMEM = 3,       /* host or device allocation failed                                        */
    POISSON_ENOKERNEL = 4,    /* poisson_solve before poisson_set_kernel                                 */
    POISSON_ECUDA = 5,        /* a CUDA call failed (sticky; text via poisson_last_error)                */
    POISSON_EARCH = 6         /* no CUDA device, or the device is not compute capability 10.x            */
};

/* Pass indices of the fused 5-pass pipeline (DESIGN.md section "Kernels"):
 * F1 = spread + 1DFFT (R2C) along the first processed axis a
 * F2 = (transpose+)spread + 1DFFT along axis b
 * F3 = spread + 1DFFT along axis c, K^F multiply, inverse 1DFFT along c, compactification
 * I2 = inverse 1DFFT along b + compactification,  I1 = inverse 1DFFT (C2R) along a + compactification */
enum { POISSON_PASS_F1 = 0, POISSON_PASS_F2 = 1, POISSON_PASS_F3 = 2, POISSON_PASS_I2 = 3, POISSON_PASS_I1 = 4 };

/* Host-side description of a plan: what the planner decided and the algorithmic work it implies.
 * Axis ids: 0 = x, 1 = y, 2 = z. */
typedef struct poisson_plan_info {
    int n[3];               /* physical grid N_x, N_y, N_z                                         */
    int bc[3];              /* boundary condition per axis                                         */
    int s[3];               /* padded transform lengths S_i = N_i * B_i  */
    int precision;          /* POISSON_FP64 / POISSON_FP32                                         */
    int order[3];           /* processing order (a, b, c): periodic axes first, free axes last
                               (PAPER.md:51), and a != x so the half spectrum S_a/2+1 never lands on
                               the contiguous axis       */
    int half_len;           /* H = S_a/2 + 1 kept after the real-to-complex pass */
    long long rows[5];      /* 1D transforms per pass (F3 counts a pencil once per direction)      */
    long long length[5];    /* transform length of each pass                                        */
    long long bytes[5];     /* algorithmic HBM bytes per pass (reads + writes, zeros never counted) */
    long long bytes_total;  /* sum of bytes[]  (= B_5 of SURVEY.md 8d)                              */
    long long workspace_bytes; /* device memory the plan owns: A1 + A2 + internal K^F + tables     */
    double fft_fraction;    /* (sum over the 3 forward steps of rows*length) / (3 S_x S_y S_z):
                               7/12 fully free, 2/3 surface, 7/12 wire */
} poisson_plan_info;

/* Planner only: fills *info for the given problem without touching any device (usable on a box
 * with no GPU).  Errors: EINVAL, EUNSUPPORTED as for poisson_plan_create. */
POISSON_API int poisson_plan_describe(int nx, int ny, int nz, const int bc[3] /* host; x,y,z */, int precision,
                          poisson_plan_info *info /* host, out */);

/* Creates a plan on the current CUDA device: validates, picks the axis order, allocates the
 * workspace (A1, A2, internal K^F) and uploads the twiddle tables.  `h` (grid spacing) is recorded
 * metadata only.  *out is set to NULL on failure.  Problem statement: PAPER.md:51.
 * Supported grids: every N_i >= 1 with padded length S_i = N_i * B_i <= 4096, odd N included ("various grid sizes",
 * PAPER.md:89).  A pass whose length is one of
 *   4 8 12 16 20 24 28 32 36 40 48 56 60 64 72 80 96 100 112 120 128 140 144 160 168 192 200 224 240 256 280 288 320 336 384 400
 *   448 480 512 576 640 768 896 1024
 * (csrc/sizes.def) runs the compiled register-engine kernel for that length; every other length (odd, factors 7, 11, ...,
 * three or more radices, primes), and the R2C / C2R pass of a grid with odd N_x, runs the any-length shared-memory
 * Stockham kernel (csrc/generic_pass.cuh) -- correct for every length, slower.  Only S_i > 4096 is refused with
 * POISSON_EUNSUPPORTED.  Errors: EINVAL, EUNSUPPORTED, ENOMEM, ECUDA, EARCH. */
POISSON_API int poisson_plan_create(poisson_plan **out /* host, out */, int nx, int ny, int nz,
                        const int bc[3] /* host; x,y,z */, double h, int precision);

/* dims = {S_z, S_y, S_x/2+1}: the shape of the K_f array poisson_set_kernel expects. */
POISSON_API int poisson_plan_kernel_dims(const poisson_plan *plan, long long dims[3] /* host, out */);

POISSON_API int poisson_plan_get_info(const poisson_plan *plan, poisson_plan_info *info /* host, out */);

/* Installs the Green's-function spectrum K^F of Eq. 3.
 *   K_f_dev: device, plan-precision REALS, C order [S_z][S_y][S_x/2+1] (numpy rfftn shape) = the
 *            unnormalised forward DFT of a real kernel K on the padded grid with K(-r) = K(r)
 *            (so K^F is real; the half not passed is K^F(-k) = K^F(k)).  16-byte aligned.
 * The library re-lays it once into the order pass F3 streams it in, folding in 1/(S_x S_y S_z)
 * ("a transposition of the associated kernel ... carried out only once").
 * Asynchronous on `stream`; K_f_dev may be freed once that work has completed. */
POISSON_API int poisson_set_kernel(poisson_plan *plan, const void *K_f_dev, void *stream);

/* The same for a kernel that is even along EVERY axis separately, K(+-x, +-y, +-z) all equal -- the free-space, wire and
 * surface Green's functions and -1/|k|^2 are -- stored at half the size (less K^F traffic).
 * Then K^F(k_a, S_b - k_b, k_c) = K^F(k_a, k_b, k_c) along the second-processed axis b, and the internal copy keeps only
 * the pencils k_b = 0 .. S_b/2: H (S_b/2 + 1) S_c reals instead of H S_b S_c.  Pass F3 reads the K^F of pencil S_b - k_b for
 * the upper half (same values, so results are bitwise those of poisson_set_kernel); its K^F traffic and the plan's largest
 * buffer halve.  K_f_dev as for poisson_set_kernel (the whole array; only k_b <= S_b/2 of it is read).  The evenness is the
 * CALLER's statement: it is not checked, and a kernel that is only inversion symmetric gives wrong results here.
 * The first call re-allocates the internal copy (device synchronisation) and drops the one-launch FUSED mode; poisson_set_kernel
 * switches back.  Register-engine F3 kernels only (else EUNSUPPORTED).  Errors: EINVAL, EUNSUPPORTED, ENOMEM, ECUDA. */
POISSON_API int poisson_set_kernel_even(poisson_plan *plan, const void *K_f_dev, void *stream);

/* The same for a real kernel K WITHOUT inversion symmetry (K(-r) != K(r): the general convolution of Eq. 2,
 * PAPER.md:37; screened / anisotropic kernels and the plane-wave local-potential convolution of PAPER.md:93), whose
 * spectrum is complex with K^F(-k) = conj K^F(k).
 *   K_f_dev: device, plan-precision COMPLEX values (interleaved re, im), C order [S_z][S_y][S_x/2+1] = numpy
 *            rfftn(K) of the real kernel on the padded grid (unnormalised forward DFT); 16-byte aligned.
 * The complex multiply runs in the any-length F3 kernel: the first call switches pass F3 of this plan to it (device
 * synchronisation, the internal K^F copy is re-allocated for complex values, the fused one-launch mode is dropped).
 * poisson_set_kernel may be called again later to go back to a real spectrum.
 * Errors: EINVAL, ENOMEM, EUNSUPPORTED, ECUDA. */
POISSON_API int poisson_set_kernel_complex(poisson_plan *plan, const void *K_f_dev, void *stream);

/* One solve (the 13 steps of PAPER.md:57-71 as 5 fused launches, or one, on `stream`; see poisson_plan_launch_mode).
 * Opt-in (POISSON_CHUNK=n planes per chunk, or POISSON_CHUNK_MB=m, read at plan creation): the three middle passes run chunk
 * by chunk of k_a planes, F1 | F2, F3, I2 per chunk | I1 = 2 + 3 * chunks launches, through an A2 buffer that holds ONE chunk
 * and therefore lives in the 126 MB L2 -- A2's four sweeps never reach HBM and the plan's workspace shrinks by most of A2
 * (fewer round trips to global memory).  Measured slower than the five whole-grid launches on B200 (the passes
 * are not DRAM bound), hence off by default; useful when device memory is the limit.
 *   rho_dev: device, plan-precision reals [nz][ny][nx], 16-byte aligned, not modified
 *   V_dev  : device, same shape; may equal rho_dev (rho is consumed before V is written)
 * Asynchronous, allocates nothing, never touches host memory.  One plan = one solve in flight
 * (the workspace is shared).  Errors: EINVAL (also: the current CUDA device is not the one the plan was created on),
 * ENOKERNEL, ECUDA. */
POISSON_API int poisson_solve(poisson_plan *plan, const void *rho_dev, void *V_dev, void *stream);

/* End-to-end variant with HOST buffers (the paper's usage: density on the host, potential wanted
 * back on the host): H2D copy of rho, poisson_solve, D2H copy of V, then a stream
 * synchronise.  rho_host / V_host: host memory (pinned for full speed), [nz][ny][nx] reals.
 * The plan owns the two device staging buffers (allocated on first use). */
POISSON_API int poisson_solve_host(poisson_plan *plan, const void *rho_host, void *V_host, void *stream);

/* Batched solves: `count` densities with the one K^F of the plan -- the paper's repeated-solve setting and its
 * stated remedy for the transfer cost, "overlap the transfer of one density with the computation of the
 * previous one".  The solves are dealt round-robin to lanes (host batches 3; device batches 3 while three sets of
 * intermediates fit the L2, else 2, or 1 when they exceed 256 MB per lane; POISSON_LANES=1..8 overrides),
 * each with its own A1 / A2 intermediates and its own internal stream, so that the tail of one solve overlaps
 * the head of the next (and, in the host variant, H2D of solve i+1 and D2H of solve i-1 overlap the passes of
 * solve i on the two copy engines).  Lanes are allocated on first use and kept by the plan (its
 * workspace_bytes grows accordingly; when device memory does not hold every lane the batch runs on the lanes that
 * fit).  With more than one lane a solve is always five launches (the cooperative fused kernel cannot overlap with
 * itself); a one-lane device batch is poisson_solve in a loop, in the plan's own launch mode.
 * Small grids (intermediates of one density <= 16 MB, i.e. up to 64^3 -> 128^3, where one solve has far fewer tiles than the
 * GPU has resident CTAs) take a different route in poisson_solve_batch: up to 32 densities per LAUNCH -- each of the
 * five launches covers the tiles of all of them, density i using slot i of a wide A1 / A2 allocation (<= 96 MB, so it
 * stays in L2) -- on the caller's stream, no lanes (POISSON_WIDE=0 disables, =n forces n per launch).
 *   rho / V : host arrays of `count` pointers; poisson_solve_batch: device buffers as in poisson_solve
 *             (rho[i] == V[i] allowed; the V[i] must not overlap each other or any other rho[j]);
 *             poisson_solve_batch_host: host buffers (pinned for overlap), [nz][ny][nx] reals each.
 * poisson_solve_batch is asynchronous: the lanes start after the work already queued on `stream`, and work
 * queued on `stream` afterwards starts after every solve of the batch.  poisson_solve_batch_host returns
 * after the last V has arrived on the host.  A plan runs ONE call at a time.
 * Errors: EINVAL (null / misaligned pointer, count < 0, current device is not the plan's), ENOKERNEL, ENOMEM, ECUDA.
 * After an error in the middle of a batch the caller's stream is still ordered after the lane work already queued. */
POISSON_API int poisson_solve_batch(poisson_plan *plan, const void *const *rho_dev /* host array of device ptrs */,
                        void *const *V_dev /* host array of device ptrs */, int count, void *stream);
POISSON_API int poisson_solve_batch_host(poisson_plan *plan, const void *const *rho_host /* host array of host ptrs */,
                             void *const *V_host /* host array of host ptrs */, int count, void *stream);
/* Densities per launch a DEVICE batch of `count` solves would use (the small-grid route above); 0 = the lane route. */
POISSON_API int poisson_plan_batch_width(const poisson_plan *plan, int count);
/* Lanes a batch of `count` solves would use (host != 0: the host variant); 0 on a null plan or count <= 0.
 * With one lane a device batch is poisson_solve in a loop (same launch mode). */
POISSON_API int poisson_plan_batch_lanes(const poisson_plan *plan, int count, int host);

/* Debug/test access to the plan's intermediates (per-pass parity).  which = 0: A1,
 * complex [.][.][.] after F1 (or after I2); which = 1: A2 after F2 / F3.  dims are the array
 * extents in memory order (z-extent, y-extent, x-extent), each axis holding N_i, S_i or H.  POISSON_EUNSUPPORTED for A2 of a
 * chunked plan (it never exists whole), as is a partial pass range in poisson_debug_run_passes there. */
POISSON_API int poisson_debug_workspace(const poisson_plan *plan, int which, void **ptr_dev /* out */,
                            long long dims[3] /* host, out */);
/* Runs passes [first, last] (POISSON_PASS_*) of a solve only; same arguments as poisson_solve. */
POISSON_API int poisson_debug_run_passes(poisson_plan *plan, const void *rho_dev, void *V_dev, void *stream,
                             int first_pass, int last_pass);

/* Per-pass device timing for the roofline report (bench.py): identical to poisson_solve, but a CUDA
 * event is recorded on `stream` before the first launch and after every launch (launches + 1 events per solve,
 * from a pool the plan owns; a chunked plan's launches are summed into their pass; at most 512 profiled solves between two reads).
 * poisson_profile_read synchronises on the recorded events, ADDS each pass's elapsed milliseconds
 * over all solves profiled since the last read into ms_sum[5], stores their number in *n_solves,
 * and resets the pool.  Errors: EINVAL, ENOKERNEL, ECUDA, ENOMEM (pool exhausted). */
POISSON_API int poisson_solve_profiled(poisson_plan *plan, const void *rho_dev, void *V_dev, void *stream);
POISSON_API int poisson_profile_read(poisson_plan *plan, double ms_sum[5] /* host, out */, int *n_solves /* host, out */);

/* How poisson_solve launches the 13 steps of PAPER.md:57-71:
 *   FIVE      five fused passes, one launch each;
 *   FIVE_PDL  the same five launches with programmatic dependent launch: a CTA that has issued the loads of its last tile
 *             lets the next pass launch, whose CTAs take the freed SM slots, build their tables and wait for the
 *             previous pass to complete (triggering at the START of a pass instead costs 10 % on the 256^3 / 512^3
 *             grids, measured: POISSON_PDL_TRIGGER=0);
 *   FUSED     ONE persistent cooperative launch: F1 | grid barrier | F2 -> F3 -> I2 as a per-plane dataflow
 *             through L2 | grid barrier | I1 (compiled for the combinations in csrc/fused_*.cu).
 *   GRAPH     the five launches as kernel nodes of one instantiated CUDA graph (one cudaGraphLaunch per solve; rho / V
 *             are patched into the F1 / I1 nodes when they change): the dependent kernels follow each other with less
 *             latency than stream launches (128^3 -> 256^3 fp64: 103.7 -> 98.7 us per solve);
 *   GRAPH_PDL the same graph with programmatic-dependent-launch edges between the kernel nodes.
 * poisson_plan_create times the available modes on scratch inputs and keeps the fastest (a few ms);
 * POISSON_TUNE=0 skips that (FIVE), POISSON_PDL=0|1, POISSON_FUSED=0|1 and POISSON_GRAPH=1 (with POISSON_PDL=1: GRAPH_PDL) force a mode.
 * poisson_plan_launch_mode reports the choice and the measured milliseconds per solve of
 * {FIVE, FIVE_PDL, FUSED, GRAPH, GRAPH_PDL} (0 where a mode was not measured). */
enum { POISSON_LAUNCH_FIVE = 0, POISSON_LAUNCH_FIVE_PDL = 1, POISSON_LAUNCH_FUSED = 2, POISSON_LAUNCH_GRAPH = 3, POISSON_LAUNCH_GRAPH_PDL = 4 };
POISSON_API int poisson_plan_launch_mode(const poisson_plan *plan, int *mode /* host, out */, double ms_per_solve[5] /* host, out */);

/* Shape of the GRAPH / GRAPH_PDL solve graph.  The five passes only couple along the axis they transform, so the graph
 * need not be a chain: with J ranges of k_a planes and R ranges of x it is
 *     F1_r -> F2_{r,j} -> F3_j -> I2_{r,j} -> I1_r          (r < R, j < J)
 * (F1 / F2 / I2 / I1 tiles of different x never exchange data, F2 / F3 / I2 tiles of different k_a neither; PAPER.md:53's
 * transposes are the only coupling), 2R + 2RJ + J kernel nodes in all.  A kernel whose successor needs only part of the
 * grid hands its SM slots to that successor while its siblings still run, which hides the ramp-up and tail of the
 * passes inside ONE solve (128^3 -> 256^3 fp64 on B200: 98.4 us as a chain, 92.3 with J = 4, 90.6 with J = R = 2).
 * poisson_plan_create times a few shapes together with the launch modes; POISSON_BRANCHES=J / POISSON_XCHAINS=R fix one.
 * When x is processed second (surface grids) the R ranges run along the other axis F1 / F2 / I2 / I1 do not couple on (the split axis o)
 * instead of x.  Ranges must hold whole tiles, else R = 1.  Outputs 1, 1 in the other modes.
 * Errors: EINVAL. */
POISSON_API int poisson_plan_graph_shape(const poisson_plan *plan, int *plane_chains /* host, out */, int *x_chains /* host, out */);

/* Number of kernel launches one poisson_solve enqueues (bench.py's gpu_launches): 5, 2 + 3 * chunks on a chunked plan, or 1
 * in FUSED mode, 2R + 2RJ + J kernel nodes for a shaped graph (poisson_plan_graph_shape). */
POISSON_API int poisson_plan_launches_per_solve(const poisson_plan *plan);

/* Measures the plain-ALU fused-multiply-add peak of the current device for the given precision
 * (independent FMA chains in registers, no memory traffic) and returns it in TFLOP/s counting an
 * FMA as 2 flops.  bench.py quotes the solve's nominal FLOP rate against this number; it is the
 * ALU bound of DESIGN.md, not a tensor-core figure.  Synchronous.  Errors: EINVAL, EARCH, ECUDA. */
POISSON_API int poisson_measure_fma_peak(int precision, double *tflops /* host, out */);

/* Environment variables.  All are read ONCE, inside poisson_plan_create (the solve path never calls getenv); none is
 * needed for normal use -- the defaults are what the plan-time timing run picks.  For users:
 *   POISSON_TUNE=0            skip the plan-time timing run (plan creation in microseconds instead of milliseconds; mode FIVE)
 *   POISSON_PDL=0|1, POISSON_FUSED=0|1, POISSON_GRAPH=1          force a launch mode (poisson_plan_launch_mode)
 *   POISSON_BRANCHES=J, POISSON_XCHAINS=R                         force the graph shape (poisson_plan_graph_shape)
 *   POISSON_CHUNK=n | POISSON_CHUNK_MB=m                          plane-chunked middle passes (poisson_solve), smaller workspace
 *   POISSON_LANES=1..8, POISSON_WIDE=0|n                          batch routes (poisson_solve_batch)
 * For the library's own experiments and tests (no stability promise; results stay correct with any value):
 *   POISSON_VARIANT, POISSON_GRID, POISSON_PREFETCH (one value, or one per pass "f1,f2,f3,i2,i1"), POISSON_LATE_TW,
 *   POISSON_PDL_TRIGGER, POISSON_FUSED_SKEW, POISSON_LANE_GRAPH=0, and POISSON_TEST_MAX_LANES=n, which makes the allocation
 *   of a batch lane beyond the n-th fail as if device memory had run out (tests of the fall-back to fewer lanes). */
POISSON_API size_t poisson_plan_workspace_bytes(const poisson_plan *plan);
POISSON_API int poisson_plan_destroy(poisson_plan *plan);

/* ---- One solve sharded over several GPUs.
 * The paper's transposes act on the reduced data set and it names direct GPU-to-GPU transfers as the way to
 * scale.  Here rho / V are distributed in slabs along the axis o (the non-x axis that is not the first
 * processed axis a: y for fully free / wire / periodic grids, z for the surface grid).  F1 transforms axis a on a rank's own
 * slab; the half spectrum then changes hands ONCE per direction, on the smallest intermediate of the pipeline (A1:
 * H x N_o x N_x complex, 33.8 MB for 128^3 -> 256^3 against 67.6 MB for A2):
 *     F1 (own slab of o)  --stores-->  every rank's plane slab  [k_a in its range][all o][x]        exchange 1
 *     F2, F3, I2 on the rank's own k_a planes (its share of K^F only)
 *     I2                  --stores-->  every rank's slab        [all k_a][its range of o][x]         exchange 2
 *     I1 (own slab of o)  ->  V
 * The exchanges are not separate copies or collectives: passes F1 and I2 store every element straight into the slab of
 * the GPU that owns it, through peer-mapped pointers (NVLink / NVSwitch peer memory), so the transfer overlaps the
 * transform tile by tile.  The caller provides the slabs (memory every peer can address: CUDA IPC / VMM / symmetric
 * memory; on one GPU any device memory) and the two cross-rank barriers:
 *     poisson_shard_forward(rho)  |  barrier A (all ranks' forward done)  |  poisson_shard_middle
 *                                 |  barrier B (all ranks' middle done)   |  poisson_shard_inverse(V)
 * each barrier ordered on `stream` (e.g. a one-element NCCL all-reduce enqueued on it).  Barrier B also protects the
 * next solve: its forward overwrites the plane slabs the middle pass has consumed by then, and its middle pass
 * overwrites the slabs pass I1 reads only after the next barrier A, which every rank enqueues after its own I1.
 * Partition: rank s of R owns [floor(T s / R), floor(T (s + 1) / R)) of T = N_o points resp. T = H planes.
 * Supported: grids whose five passes all run the compiled register-engine kernels, even N_x, R <= min(N_o, H, 32);
 * else POISSON_EUNSUPPORTED.  Results are bitwise those of poisson_solve (same kernels, same arithmetic per pencil), with one
 * exception: shard plans always take a length's default factorisation, while poisson_solve runs passes F2 / I2 of length 192 in
 * fp64 in a second, faster one (12 x 16) -- on grids with S_b = 192 the two agree to rounding (1e-15), not bit for bit. */
typedef struct poisson_shard_info {
    int rank, nranks;
    int split_axis;         /* o: rho / V are distributed along this axis (1 = y, 2 = z)                          */
    int plane_axis;         /* a: between the exchanges the half spectrum k_a = 0 .. H-1 of this axis is distributed */
    int o0, o1;             /* this rank's slab: o0 <= o < o1                                                       */
    int k0, k1;             /* its planes: k0 <= k_a < k1                                                           */
    long long local_dims[3];   /* shape of the rank's rho / V, C order [z][y][x]                                    */
    long long mid_dims[3];     /* shape of its exchange slab 1 (complex), C order: A1 with axis a -> k1 - k0        */
    long long back_dims[3];    /* shape of its exchange slab 2 (complex), C order: A1 with axis o -> o1 - o0        */
    long long mid_bytes, back_bytes;   /* sizes of the two slabs the caller must provide for this rank              */
    long long sent_bytes[2];   /* bytes this rank stores into OTHER ranks' slabs in exchange 1 / exchange 2          */
    long long workspace_bytes; /* device memory the plan itself owns (A2 of its planes, its share of K^F, tables)   */
} poisson_shard_info;

/* Planner only (no device needed).  Errors: EINVAL, EUNSUPPORTED. */
POISSON_API int poisson_shard_describe(int nx, int ny, int nz, const int bc[3], int precision, int rank, int nranks,
                                       poisson_shard_info *info /* host, out */);
/* Plan of rank `rank` of `nranks` for the GLOBAL grid nx, ny, nz on the current device.  A shard plan only takes the
 * poisson_shard_* calls (plus poisson_plan_kernel_dims / _destroy); poisson_solve on it returns EINVAL. */
POISSON_API int poisson_shard_plan_create(poisson_plan **out, int nx, int ny, int nz, const int bc[3], double h, int precision,
                                          int rank, int nranks);
POISSON_API int poisson_shard_get_info(const poisson_plan *plan, poisson_shard_info *info /* host, out */);
/* mid_of_rank[s] / back_of_rank[s]: device pointers, valid on THIS device, to rank s's exchange slabs (host arrays of
 * nranks pointers; entry [rank] is the rank's own slab).  32-byte aligned (passes F1 / I2 store 256-bit pairs into them), else
 * EINVAL; EINVAL also when the current device is not the plan's.  The plan keeps the pointers, not the memory. */
POISSON_API int poisson_shard_set_slabs(poisson_plan *plan, void *const *mid_of_rank /* host */, void *const *back_of_rank /* host */);
/* K_f_dev: the WHOLE spectrum [S_z][S_y][S_x/2+1] as for poisson_set_kernel; only the rank's planes are kept. */
POISSON_API int poisson_shard_set_kernel(poisson_plan *plan, const void *K_f_dev, void *stream);
/* The three stages of one sharded solve (asynchronous on `stream`; the caller enqueues the barriers between them).
 * rho_local_dev / V_local_dev: the rank's slab, plan precision, C order local_dims.  Errors: EINVAL, ENOKERNEL, ECUDA. */
POISSON_API int poisson_shard_forward(poisson_plan *plan, const void *rho_local_dev, void *stream);
POISSON_API int poisson_shard_middle(poisson_plan *plan, void *stream);
POISSON_API int poisson_shard_inverse(poisson_plan *plan, void *V_local_dev, void *stream);

/* ---- One solve for callers that cannot allocate device memory.
 * Everything above needs a plan, and a plan is made of cudaMalloc'ed buffers (intermediates, its copy of K^F, twiddle
 * tables).  Some programs cannot give it that: a simulation code that took all of the GPU's memory for its own pool at
 * start-up, so that a cudaMalloc made by a library it calls simply fails; a process held to a fixed memory budget by
 * its job scheduler; or an inner loop (an SCF cycle, a time step) in which the device-wide synchronisation hidden in
 * cudaMalloc / cudaFree, or an out-of-memory error at step 10 000, is not acceptable.  For them this ONE call does a
 * whole solve -- K^F re-layout, F1, F2, F3, I2, I1: the same kernels, the same kernel choice, hence the same bits as
 * poisson_plan_create + poisson_set_kernel + poisson_solve -- and calls no cudaMalloc, cudaFree or other allocating
 * routine.  Its scratch is a fixed array of POISSON_STATIC_SCRATCH_BYTES that is part of the library image: every GPU
 * on which the process uses this library holds that much from the moment the library's code is loaded there until the
 * process exits, whether or not this function is ever called.
 *   nx, ny, nz, bc, precision: the problem, as for poisson_plan_create (no h: it is metadata there)
 *   K_f_dev : device, the spectrum exactly as poisson_set_kernel takes it (real, even kernel; [S_z][S_y][S_x/2+1]);
 *             it is re-laid on EVERY call -- there is no plan to remember it -- which costs one extra sweep over K^F
 *   rho_dev, V_dev: device, as for poisson_solve (16-byte aligned, rho_dev == V_dev allowed)
 * Limit: tables (576 KiB) + A1 + A2 + the K^F copy must fit the array.  32^3 -> 64^3 free (3.3 MB) and 64^3 -> 128^3
 * free in fp64 (21.9 MB) fit, 96^3 -> 192^3 fp64 does not; a grid that does not fit is refused with POISSON_EUNSUPPORTED
 * and poisson_last_error() says how many bytes it would need.  Nothing is launched in that case.
 * Sharing: there is one array per GPU and every call on that GPU uses it.  Two calls whose GPU work can overlap (two
 * streams, two host threads with their own streams) overwrite each other's intermediates: order them yourself (same
 * stream, or an event between them).  The host side is serialised by a mutex.  The array keeps what the last call left
 * in it; no call depends on that (each call writes every byte before it reads it -- nothing has to be zeroed), except
 * the twiddle tables, which are kept on purpose and re-uploaded only when a transform length or the precision changes.
 * First call on a device: resolves the array's device address (cudaGetSymbolAddress, with that device current) and
 * checks the architecture; the first call for a new set of transform lengths copies their tables from ordinary host
 * memory, which makes the host wait for the work already queued on `stream`.  Make that first call outside any
 * stream capture.  Asynchronous otherwise.  Errors: EINVAL, EUNSUPPORTED (also: over the limit), ECUDA, EARCH. */
#define POISSON_STATIC_SCRATCH_BYTES (32u << 20)
POISSON_API int poisson_solve_static(int nx, int ny, int nz, const int bc[3] /* host; x,y,z */, int precision,
                                     const void *K_f_dev, const void *rho_dev, void *V_dev, void *stream);

POISSON_API const char *poisson_status_string(int status);
/* Text of the last CUDA error seen by this thread's most recent failing call ("" if none). */
POISSON_API const char *poisson_last_error(void);
/* "sm_100a" etc.: the architecture the kernels were compiled for. */
POISSON_API const char *poisson_build_arch(void);

#ifdef __cplusplus
}
#endif
#endif /* POISSON_B200_H */
