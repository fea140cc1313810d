/* lrmd.h — C ABI of the B200 (sm_100a) long-range molecular-dynamics hot path.
 *
 * What it computes: the data-parallel hot path of arXiv 1212.0262 (T. M. Rocha Filho,
 * "Molecular dynamics for long-range interacting systems on Graphic Processing Units"):
 * force evaluation, fused kick/drift updates and energy sums of the fourth-order symplectic
 * integrator for three N-body models of unit-mass particles (PAPER.md = /root/reference/PAPER.md):
 *
 *   LRMD_HMF     H = 1/2 sum p_i^2 + (1/N) sum_{i<j} [1 - cos(th_i - th_j)]            PAPER.md:36 eq.(2)
 *   LRMD_RING    H = 1/2 sum p_i^2 - (1/N) sum_{i<j} 1/(sqrt2 sqrt(1 - cos(th_i-th_j) + eps))   PAPER.md:29 eq.(1)
 *   LRMD_GRAV2D  H = 1/2 sum (px_i^2 + py_i^2) + (1/N) sum_{i<j} log[(x_i-x_j)^2 + (y_i-y_j)^2 + eps]   PAPER.md:40 eq.(3)
 *
 * Forces are f = -dH/dq:
 *   HMF     f_i = cos(th_i) My - sin(th_i) Mx, (Mx,My) = (1/N) sum (cos th_j, sin th_j)   PAPER.md:73-77 eqs.(6)-(7)
 *   RING    f_i = -(1/(2 sqrt2 N)) sum_j (s_i c_j - c_i s_j) / (1 + eps - c_i c_j - s_i s_j)^(3/2)
 *           PAPER.md:88,97 eqs.(8)-(9); the sign is that of -dH/dtheta (eq.(8) prints the opposite
 *           sign; reading G1)
 *   GRAV2D  F_i = -(2/N) sum_j (r_i - r_j) / (|r_i - r_j|^2 + eps)                       PAPER.md:110, from eq.(3)
 *
 * One time step is Yoshida's composition, eq.(4) and the 12-step listing
 * PAPER.md:54-62 (readings G2-G4): with f = F(q) cached,
 *   p += B0 dt f; q += D0 dt p; f = F(q);  p += B1 dt f; q += D1 dt p; f = F(q);
 *   p += B1 dt f; q += D0 dt p; f = F(q);  p += B0 dt f            (f is kept for the next step)
 * i.e. three force evaluations per step, 3n+1 for n steps from a fresh state.
 *
 * Conventions
 *   - All array arguments are DEVICE pointers to contiguous fp64 arrays of length N on the
 *     current CUDA device, 16-byte aligned, owned by the caller.  The only HOST pointers are
 *     `out`, `bytes` and the const char* returned by lrmd_strerror.
 *   - The library never allocates device memory: scratch comes from lrmd_set_workspace().
 *   - Work is enqueued on the given CUDA stream (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream) and the call returns without synchronising, except where stated.
 *   - Every call returns LRMD_OK (0) or a negative error code; nothing throws, prints or exits.
 *   - Calls on one context are not thread-safe; different contexts are independent.
 *   - Results are bitwise reproducible run to run for fixed (model, N, eps, options): all
 *     reductions use fixed trees and there are no floating-point atomics.
 *   - Streams: calls on one context must be issued to one stream at a time (or be ordered by the caller's
 *     events); different contexts may run on different streams concurrently.  No call waits for, or
 *     enqueues on, any other stream (tests/test_gpu_streams.py).
 *   - Capturing calls in a CUDA graph: lrmd_step (substage kernels: LRMD_OPT_HMF_VARIANT 0-2; all pair
 *     kernels), lrmd_forces and lrmd_energy enqueue plain kernel launches only, so the caller may capture them
 *     on a capturing stream PROVIDED one eager lrmd_step (and one eager call of whatever else is captured) ran
 *     on the context before: that caches the force and raises the kernels' shared-memory limits, so the
 *     captured sequence is the steady-state one.  Every replay advances the bound state by the captured
 *     steps.  The library's own graph replay (LRMD_OPT_GRAPH) stands aside while the stream is capturing.
 *     Not for capture: lrmd_set_workspace, lrmd_step_host, lrmd_kernel_time (they synchronise) and contexts
 *     with LRMD_OPT_KERNEL_TIMING on (event records); the resident HMF kernels (variants 3, 4) are untested.
 */
#ifndef LRMD_H_
#define LRMD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lrmd_ctx lrmd_ctx;

enum { LRMD_HMF = 0, LRMD_RING = 1, LRMD_GRAV2D = 2 };

enum {
    LRMD_OK = 0,
    LRMD_EINVAL = -1,        /* bad argument (NULL, wrong NULL pattern, N < 1, eps <= 0 ...)  */
    LRMD_ESTATE = -2,        /* state or workspace not set                                     */
    LRMD_ECUDA = -3,         /* a CUDA call failed; see lrmd_last_cuda_error                   */
    LRMD_EUNSUPPORTED = -4,  /* valid request this build does not implement                    */
    LRMD_ECOLL = -5,         /* a collective callback of a sharded context returned non-zero   */
    LRMD_ETOOBIG = -6        /* lrmd_hmf_forces_static: N exceeds LRMD_STATIC_MAX_N (the built-in scratch array) */
};

/* lrmd_set_option keys */
enum {
    LRMD_OPT_PAIR_PRECISION = 0, /* 0 = fp64 pair arithmetic (default); 1 = fp32 pair arithmetic with chunked
                                    fp32 -> fp64 accumulation: GRAV2D on positions rounded to
                                    fp32, RING on (cos, sin)(theta / 2) rounded to fp32 (half-angle form: eq.(9)'s
                                    denominator cancels to ~eps and would lose the 1e-5 tolerance in fp32); needs
                                    eps >= 1e-30; HMF: LRMD_EUNSUPPORTED                                            */
    LRMD_OPT_PAIR_CTAS = 1,      /* pair models: number of CTAs G the flattened (i-tile, j) space is divided
                                    into, equal shares (0 = choose from N: 148 x resident CTAs x waves)  */
    LRMD_OPT_GRAPH = 2,          /* HMF substage kernels: 1 = lrmd_step replays a captured CUDA graph of 8 steps
                                    (24 kernel nodes) for the steady-state steps, 0 = plain launches, -1 = choose (1;
                                    never for shards, the resident kernels, or while kernel timing is on)          */
    LRMD_OPT_HMF_GRID = 3,       /* HMF: number of CTAs of the fused substage kernel (0 = choose)      */
    LRMD_OPT_KERNEL_TIMING = 4,  /* 1 = bracket every launch of the model's dominant kernel (HMF: the fused
                                    substage kernel; RING/GRAV2D: the pair-force kernel) with a CUDA event
                                    pair on the launching stream; read with lrmd_kernel_time.  Turns CUDA-graph
                                    replay off while set.  Measurement aid: results are unchanged.          */
    LRMD_OPT_HMF_VARIANT = 5,    /* HMF: 0 = register-prefetch substage kernel, 1-2 = TMA-staged substage kernel
                                    shapes, 3 = cluster-resident kernel (N <= 20,480: state in registers of one
                                    thread-block cluster, all n steps of a call in one launch), 4 = grid-resident kernel
                                    (N <= 1,070,336: state in the shared memory of one CTA per SM, all n steps of a call
                                    in one cooperative launch, a grid barrier per substage; if the device refuses the cooperative
                                    launch — cudaErrorCooperativeLaunchTooLarge, NotSupported, InvalidValue or
                                    InvalidConfiguration, e.g. under MPS with fewer SMs — the context switches to the substage
                                    kernels for good and lrmd_get_option shows the variant then in use; any other CUDA error
                                    is returned as LRMD_ECUDA); -1 = choose from N (3 up to 20,480, 4 up to 1,070,336,
                                    1 beyond; shards: 0 below 1e6, else 1)                                                  */
    LRMD_OPT_PAIR_VARIANT = 6,   /* pair models: launch shape of the pair kernels (-1 = choose).  Ordered kernels:
                                    0 = 128 threads x 4 rows, 1 = 128 x 8, 2 = 256 x 4.  Symmetric and band kernels:
                                    0 = 4 rows per lane, 1 (and 2) = 8; fp32 band kernel: 2 = 16 rows per lane            */
    LRMD_OPT_PAIR_SLOTS = 7,     /* read-only (lrmd_get_option): partial force rows per particle          */
    LRMD_OPT_PAIR_SYMMETRIC = 8, /* pair models: force kernels that evaluate every UNORDERED pair once and add +f / -f to
                                    both particles (the paper declines this): 1 = warp-level
                                    kernel (one j-side scratch row per 32R-particle tile; fp64 and, GRAV2D, fp32 pairs),
                                    2 = band kernel (fp64, and GRAV2D fp32 pairs; both sides' sums kept on chip over blocks of 8 x 32R
                                    particles, one launch for any N; scratch about 40 N doubles per component with the default band height —
                                    673 MB at config 5, N = 2^20 — see lrmd_workspace_bytes);
                                    0 = every ordered pair (the paper's scheme); -1 = choose (1 for 2048 <= N < 49,152,
                                    2 beyond, 0 if the context is a shard).  get: the kernel in use.  With 1
                                    LRMD_OPT_PAIR_CTAS counts warps (workers) per launch, with 2 CTAs.                */
    LRMD_OPT_PAIR_SYM_TILES = 9, /* symmetric kernel: i-tiles per launch (0 = as many as keep the j-side scratch rows,
                                    N doubles per tile and component, within 1 GiB); get: the value in use            */
    LRMD_OPT_PAIR_FUSE_UPDATE = 10, /* symmetric kernel, one launch per force evaluation: 0 = separate update kernel,
                                    1 / -1 = the kick / drift that follows a force evaluation runs inside its fold
                                    kernel (same arithmetic, bit-identical results); get: whether it is in use       */
    LRMD_OPT_PAIR_SYM_EXCHANGE = 11, /* symmetric fp64 kernel: how the j-packet (position + collected force) meets the lanes:
                                    0 = it travels around the warp by shuffles, 1-3 = it lives in a per-warp shared-memory
                                    buffer (register budget for 2, 3, 4 resident CTAs per SM); -1 = choose (3).  fp32 band
                                    kernel (GRAV2D, pair precision 1): 0 = the j-side sum of a slot is an fp32 packet that
                                    travels with the slot by shuffles and joins the fp64 sum once per 32-step visit (fp32
                                    over 32 R terms), 1-3 = it joins the slot's fp64 sum in shared memory every step (fp32
                                    over R terms); -1 = choose (0).  Results differ between 0 and 1-3 in the rounding of
                                    the j-side sums only.                                                             */
    LRMD_OPT_PAIR_BAND_HEIGHT = 12  /* band kernel: I-blocks per band.  0 = choose: the tallest band whose i-side scratch rows,
                                    which all CTAs cycle through, stay within 80 MB of the L2 (16 at config 5); only when
                                    that choice would need more than 1 GiB of rows, the height that minimises the scratch
                                    (N = 3e6: 24).  get: the value in use                                               */
};

/* Create a context for `model` (LRMD_HMF | LRMD_RING | LRMD_GRAV2D) with N >= 1 particles.
 * eps: softening of eqs.(1),(3); ignored for HMF; must be finite and > 0 for RING and GRAV2D
 * (the pair kernels include the j = i term, which is exactly zero only for eps > 0 — the
 * paper's tile loop does the same).  The library owns *out (host memory only). */
int lrmd_create(lrmd_ctx** out, int model, int64_t N, double eps);

/* Free the context (host memory only; device buffers belong to the caller). NULL is LRMD_EINVAL. */
int lrmd_destroy(lrmd_ctx* ctx);

/* Scratch needed for the current options: partial sums, the packed j-stream (cos,sin) or (x,y)
 * of PAPER.md:100, partial forces, device scalars.  Query, allocate `*bytes` on the device
 * (256-byte aligned), then bind it.  Changing an option that alters the size returns the
 * context to "workspace not set".  A context that uses a symmetric or band pair kernel keeps work tables
 * in the workspace which every resolving call rebuilds: there ANY lrmd_set_option (except KERNEL_TIMING,
 * PAIR_FUSE_UPDATE and PAIR_SYM_EXCHANGE) and any lrmd_set_shard returns the context to "workspace not
 * set", even if the size did not change — call lrmd_set_workspace again (the next call otherwise returns
 * LRMD_ESTATE).  The contents are private to the library. */
int lrmd_workspace_bytes(const lrmd_ctx* ctx, size_t* bytes);
/* lrmd_set_workspace copies the small work tables of the symmetric / band pair kernels (a few KB to a few MB, built on
 * the host when the options were resolved) into the workspace with cudaMemcpyAsync on cuda_stream and SYNCHRONISES
 * that stream before returning (the host tables may be rebuilt by the next lrmd_set_option).  For the other contexts
 * (HMF, ordered pair kernels) it touches no device memory and does not synchronise. */
int lrmd_set_workspace(lrmd_ctx* ctx, void* device_ptr, size_t bytes, void* cuda_stream);

/* Bind the state arrays, updated IN PLACE by lrmd_step.
 *   HMF, RING: (theta, p, NULL, NULL);   GRAV2D: (x, y, px, py).
 * Any other NULL pattern is LRMD_EINVAL.  Binding invalidates the cached force: call it again
 * after modifying the arrays yourself.  Angles are never wrapped (reading G8). */
int lrmd_set_state(lrmd_ctx* ctx, double* a0, double* a1, double* a2, double* a3);

/* Advance n >= 0 full steps of size dt (may be negative) of eq.(4).  n = 0 is a no-op. */
int lrmd_step(lrmd_ctx* ctx, int64_t n, double dt, void* cuda_stream);

/* End-to-end variant with HOST buffers (pinned memory recommended), same NULL pattern as lrmd_set_state:
 * copies h_* into the bound device state arrays (cudaMemcpyAsync on the stream; this invalidates the
 * cached force), advances n steps, copies the state back into h_* and SYNCHRONISES the stream before
 * returning.  The device state arrays must have been bound with lrmd_set_state. */
int lrmd_step_host(lrmd_ctx* ctx, double* h_a0, double* h_a1, double* h_a2, double* h_a3, int64_t n, double dt,
                   void* cuda_stream);

/* Write the force at the current positions: f0 = f (HMF, RING; f1 must be NULL) or
 * (f0, f1) = (fx, fy) (GRAV2D).  Uses the cached force if valid, else evaluates and caches it. */
int lrmd_forces(lrmd_ctx* ctx, double* f0, double* f1, void* cuda_stream);

/* Write out4[0..3] = {K, V, a, b} (DEVICE pointer to 4 doubles):
 *   K = 1/2 sum p^2;  V = the potential energy of eqs.(1)-(3)
 *   (HMF: V = (N/2)(1 - Mx^2 - My^2), eq.(5); RING, GRAV2D: O(N^2) pair sum over i<j);
 *   (a, b) = (Mx, My) for HMF, (sum p, 0) for RING, (sum px, sum py) for GRAV2D. */
int lrmd_energy(lrmd_ctx* ctx, double* out4_device, void* cuda_stream);

/* Advance n >= 0 steps and record the observables the paper plots against time (K, V and the energy
 * error derived from them, PAPER.md:136 and Figs. 3-6; "compute any properties of interest", listing
 * step 12): out_device (DEVICE pointer, 4 * (n / every + 1) doubles) receives the
 * lrmd_energy record {K, V, a, b} of the initial state followed by one record after every `every`-th
 * step (every >= 1).  Steps left over after the last record (n % every) are taken without a record.
 * Asynchronous on the stream, like lrmd_step. */
int lrmd_step_observe(lrmd_ctx* ctx, int64_t n, double dt, int64_t every, double* out_device, void* cuda_stream);

/* Multi-GPU sharding (PAPER.md:82 for HMF, PAPER.md:112-124 for the pair models).  One process
 * per GPU; each creates its context with N = the number of particles it OWNS and declares here that they are the
 * global indices i0 .. i0 + N - 1 of N_total.  State arrays, forces and lrmd_step_host buffers hold the owned
 * particles only.  The exchange steps are the caller's collectives (NCCL through torch.distributed in the Python
 * binding), called by the library on the stream between its kernels:
 *   HMF          after every reduction: allreduce(device pointer to this rank's (sum cos, sum sin), 2, stream, user)
 *                must sum the 2 doubles over all ranks in place (each GPU "computes the magnetization
 *                components for its corresponding number of particles, and their sum give the total");
 *   RING/GRAV2D  after every drift: allgather(device pointer to the packed j-stream of ALL N_total particles,
 *                elem_bytes, i0, N, N_total, stream, user) — this rank's N elements are already in place at element
 *                offset i0; the callback must fill in the other ranks' (each GPU stores half of the momenta
 *                and forces "but all the particle position coordinates").
 * A callback returns 0 on success.  lrmd_energy on a shard returns this rank's part of K, of V (pair models: rows
 * owned x all j, halved) and of the momentum sums — add them over ranks; HMF's V, Mx, My are already global.
 * N_total = N (a single shard) restores the unsharded path.  Changes the workspace size. */
typedef int (*lrmd_allreduce_fn)(void* device_doubles, int64_t count, void* cuda_stream, void* user);
typedef int (*lrmd_allgather_fn)(void* device_all, int64_t elem_bytes, int64_t i0, int64_t n_local, int64_t n_total,
                                 void* cuda_stream, void* user);
int lrmd_set_shard(lrmd_ctx* ctx, int64_t N_total, int64_t i0, lrmd_allreduce_fn allreduce, lrmd_allgather_fn allgather,
                   void* user);

/* HMF force for callers that have no way to provide scratch memory.
 *
 * Every other call above needs a workspace that the caller allocates (lrmd_workspace_bytes -> cudaMalloc or a torch
 * tensor -> lrmd_set_workspace).  Some callers cannot do that: a plug-in whose host application grabbed all of the
 * device memory for its own pool at start-up and hands the plug-in nothing but input and output pointers; a routine
 * called from inside a latency-critical loop, where cudaMalloc / cudaFree are off limits because they stall the whole
 * device; a C interface that was fixed before a workspace argument could be added.  This one call serves them.  It
 * computes, for N particles of the HMF model,
 *     f_i = cos(theta_i) My - sin(theta_i) Mx,  (Mx, My) = (1/N) sum_j (cos theta_j, sin theta_j)      PAPER.md:73-77 eqs.(6)-(7)
 * exactly as lrmd_forces does, needs no context and no workspace, and calls no cudaMalloc, cudaFree or any other
 * allocating routine — neither on the first call nor later.  Its scratch, one (sum cos, sum sin) pair per CTA of the
 * reduction kernel, lives in an array built into the library: LRMD_STATIC_SCRATCH_BYTES (64 KiB) of device memory,
 * held on every GPU that loads liblrmd.so until the process exits, whether or not this call is ever used.
 *
 *   theta_device  DEVICE, N doubles, 8-byte aligned, read only            f_device  DEVICE, N doubles, written
 *   N             1 .. LRMD_STATIC_MAX_N (4,194,304 = 4096 CTA sums x 1024 particles each).  A larger N does not fit
 *                 the built-in array and is refused with LRMD_ETOOBIG before anything is launched; use a context.
 *   cuda_stream   the two kernels (per-CTA sums, then the forces) are enqueued on it; the call does not synchronise
 *   cuda_error_host  HOST, may be NULL: receives the cudaError_t (as int) behind an LRMD_ECUDA return, else 0
 *
 * The current device must be the one that owns theta_device, f_device and the stream.
 * First call on a device: the library looks up the device address of its scratch array once per device
 * (cudaGetSymbolAddress; the array's name is not a usable pointer in host code) and remembers it; this lookup is
 * thread-safe.  Make that first call on each device before starting any stream capture.
 * All calls on a device share the one array and it keeps whatever the previous call left there.  Nothing in it has to
 * start at zero: each call overwrites every entry it later reads.  Calls issued to the SAME stream are ordered and
 * safe.  Calls that can run at the same time on one GPU (different streams, different host threads, different
 * processes each have their own copy — only calls within one process share it) overwrite each other's sums and
 * return wrong forces: serialise them yourself.
 * Other returns: LRMD_EINVAL (NULL or misaligned pointer, N < 1), LRMD_EUNSUPPORTED (device ordinal >= 64). */
#define LRMD_STATIC_MAX_N 4194304
#define LRMD_STATIC_SCRATCH_BYTES 65536
int lrmd_hmf_forces_static(const double* theta_device, double* f_device, int64_t N, void* cuda_stream,
                           int* cuda_error_host);

/* Set an option (keys above).  Unknown key or bad value: LRMD_EINVAL. */
int lrmd_set_option(lrmd_ctx* ctx, int key, int64_t value);
/* Read back an option as resolved for this context (e.g. the j-split chosen from N). */
int lrmd_get_option(const lrmd_ctx* ctx, int key, int64_t* value);

/* Number of kernel launches (graph kernel nodes counted individually) enqueued by this context
 * since creation: the caller's evidence that the CUDA path ran. */
int lrmd_launch_count(const lrmd_ctx* ctx, int64_t* launches);

/* With LRMD_OPT_KERNEL_TIMING on: waits for the recorded events, writes the summed device time (ms)
 * of the dominant kernel's launches since the last call (or since the option was set) and their
 * number to the two HOST pointers, and resets the accumulation.  At most 16384 launches are recorded
 * between reads; later ones run untimed. */
int lrmd_kernel_time(lrmd_ctx* ctx, double* ms_total_host, int64_t* launches_host);

/* The cudaError_t (as int) of the last failed CUDA call on this context, 0 if none. */
int lrmd_last_cuda_error(const lrmd_ctx* ctx);

/* Static string for an error code. Never NULL. */
const char* lrmd_strerror(int code);

/* Yoshida coefficients used by lrmd_step: out4_host = {B0, B1, D0, D1} (HOST pointer). */
int lrmd_coefficients(double* out4_host);

/* Diagnostic (HOST pointers, runs on the CPU, no GPU needed): evaluates the library's own fp64
 * sincos arithmetic (csrc/trig.cuh, the routine the HMF and Ring kernels inline) on n host values,
 * so that its accuracy can be checked against a multiprecision reference without a GPU. */
int lrmd_host_sincos(const double* x_host, int64_t n, double* s_host, double* c_host);

/* Diagnostic (measurement aid, not on the hot path; SYNCHRONISES the stream): FP64 issue-rate microbenchmark, the
 * measured counterpart of the derived `alu` roofline denominator 148 SMs x 64 FP64 lanes x clock that bounds the
 * pair kernels (SURVEY.md section 7 hard part 8).  Every thread of 148 x warps_per_sm warps
 * (warps_per_sm a multiple of 4, 4..64) runs `iters` rounds of 16 independent chains of op (0 = DFMA with two
 * operands shared by all chains, 1 = DMUL, 2 = DADD, 3 = DFMA on three private registers, 4 = DFMA with one shared
 * operand, 5 = DFMA a*a+c, 6 = DFMA with an immediate addend) and, per round, extra_per_16 (0, 2, 4, 8 or 16)
 * instructions of class mix (0 none, 1 integer LOP3, 2 MUFU.RCP64H, 3 SHFL, 4 LDS.64, 5 MUFU.RCP64H seed + the DFMA
 * that consumes it, 6 MOV, 7 STS.64), op = 0 only for mix != 0.
 * scratch_device: DEVICE, 256-byte aligned, at least 148 x warps_per_sm x 32 x 8 + 148 x warps_per_sm x 4 + 1024
 * bytes, caller-owned.  out4_host (HOST) = {FP64 instructions per second (thread level), SM clock held in MHz
 * (clock64 over globaltimer inside the kernel), FP64 lanes busy per clock per SM, kernel milliseconds}.
 * Unknown combination: LRMD_EUNSUPPORTED.  Needs no context. */
int lrmd_fp64_peak(int op, int mix, int extra_per_16, int warps_per_sm, int iters, void* scratch_device,
                   size_t scratch_bytes, double* out4_host, void* cuda_stream);

/* Diagnostic (HOST pointers, runs on the CPU, no GPU needed): the work partition of the pair kernels
 * (RING, GRAV2D) for the current options.  The N x N pair rectangle (every ordered pair is computed,
 * PAPER.md:108; tiles after PAPER.md:100-106) is cut into i-tiles; the flattened (i-tile, j) space is
 * divided into LRMD_OPT_PAIR_CTAS equal contiguous ranges, one per CTA.  Writes the segments of CTA
 * `cta` as rows {tile, jbeg, jend, slot} (4 int64 each, at most max_seg rows) and their number to
 * *nseg_host: the CTA adds the pairs (i in tile) x (jbeg <= j < jend) into partial force row `slot`. */
int lrmd_pair_partition(const lrmd_ctx* ctx, int64_t cta, int64_t* seg4_host, int64_t max_seg, int64_t* nseg_host);

/* Diagnostic (HOST pointers, no GPU needed): the work partition of the band kernel (LRMD_OPT_PAIR_SYMMETRIC = 2).
 * Particles are grouped into I-blocks of IB rows and these into bands; band A's work is every pair (i in the band,
 * j >= the band's first row), cut into column ranges ("pieces").  *n_pieces_host (if not NULL) receives the number of
 * pieces (0 if the band kernel is not in use); out8_host (if not NULL) receives, for piece `piece`,
 * {band, c0, c1 (columns [32 c0, 32 c1)), owning worker, first I-block of the band, I-blocks in the band, IB, workers}. */
int lrmd_pair_band_partition(const lrmd_ctx* ctx, int64_t piece, int64_t* out8_host, int64_t* n_pieces_host);

/* Diagnostic (HOST pointers, no GPU needed): the work table of the symmetric pair kernel (LRMD_OPT_PAIR_SYMMETRIC).
 * Work units are (i-tile, chunk of 32 j) pairs with chunk >= tile * (tile size / 32), in tile-major order; each
 * launch (batch of consecutive tiles) divides its units evenly over its workers (warps).  *n_workers_host (if not
 * NULL) receives the total number of workers over all launches (0 if the symmetric kernel is not in use);
 * out5_host (if not NULL) receives {tile, chunk, units, launch, tile size} of worker `worker`. */
int lrmd_pair_sym_partition(const lrmd_ctx* ctx, int64_t worker, int64_t* out5_host, int64_t* n_workers_host);

#ifdef __cplusplus
}
#endif
#endif /* LRMD_H_ */
