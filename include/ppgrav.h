/* ppgrav.h -- C ABI of libppgrav: direct particle-particle (PP) gravity on one NVIDIA B200 (sm_100a).
 *
 * The library implements the hot path of Khrapov, Khoperskov & Khoperskov, "New features of parallel
 * implementation of N-body problems on GPU" (2018); citations are PAPER.md:<line> of /root/reference/PAPER.md.
 *
 *   pp_forces      eq. (1)-(2), PAPER.md:41-48   a_i = -G sum_{j != i} m_j (r_i - r_j) / (|r_i - r_j|^2 + delta^2)^{3/2}
 *                                                Phi_i = -G sum_{j != i} m_j / (|r_i - r_j|^2 + delta^2)^{1/2}
 *   pp_step_kdk    eqs. (5)-(7), PAPER.md:67-92  kick-drift-kick leapfrog, one gravity solve per step
 *   pp_invariants  eqs. (8)-(10), PAPER.md:148-156  E = K + W, P, L, centre of mass, total mass
 *
 * Conventions common to every call
 *   - Plain C, no exceptions.  Every function returns an int status: PP_OK (0) or a negative PP_E* code;
 *     pp_last_error() then returns a human-readable message for the calling thread.
 *   - Unless the name ends in _host, every data pointer is a DEVICE pointer on the current CUDA device, owned by
 *     the caller; the library never frees or retains it.  Work is enqueued on `stream` (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream) and the call returns without synchronising.
 *   - _host variants take HOST pointers (pageable or pinned), copy in, run the same kernels, copy out and
 *     synchronise `stream` before returning.
 *   - Layout: pos, vel, acc are row-major [N,3]; mass, pot are [N]; element type float (PP_F32) or double
 *     (PP_F64, PP_MIXED) according to `precision`; pointers must be aligned to the element size.  No padding is
 *     required.
 *   - delta is the Plummer softening length of PAPER.md:48 (delta >= 0).  delta == 0 is legal, and so is any tiny
 *     delta: when delta^2 < 1e-20 (PP_F32, PP_MIXED) or < 1e-200 (PP_F64) the guarded kernels run, in which a pair
 *     whose softened squared distance r^2 + delta^2 is at or below that threshold -- j == i, coincident bodies,
 *     padding -- contributes nothing (its r^-3 would overflow).  Above the threshold no pair is dropped.
 *   - G multiplies the finished sums once (acc = G * sum), not every pair.
 *   - Results are bit-reproducible run to run for the same N, plan and device (no floating-point atomics).
 *   - The library keeps a per-device workspace (packed copy of the bodies, split-j partial sums) that grows on
 *     demand and is freed by pp_release().  Its reuse is stream-ordered: calls on one stream follow each other as
 *     usual; a call issued on a DIFFERENT stream than the previous call on that device first waits, on the device,
 *     for the previous call's work (an event wait, no host block).  Calls from several host threads are serialised
 *     by a mutex.  So concurrent use from several streams is safe but does not overlap.
 *   - There is no CPU fallback: without a CUDA device every compute call returns PP_ECUDA.
 */
#ifndef PPGRAV_H_
#define PPGRAV_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PPGRAV_VERSION 200 /* 0.2.0 */

/* precision */
#define PP_F32 0
#define PP_F64 1
/* Extension, not in the paper (motivated by its conclusion): FP64 state and
 * FP64 time integration, FP32 pair sweep.  Every array is double; each gravity solve rounds the positions and masses
 * to FP32, runs the PP_F32 sweep (same accuracy as PP_F32: ~1e-7 of |a_i|), and adds and scales its partial sums in
 * FP64.  What it removes is the rounding of r += dt*v and v += dt/2*a in FP32, at the speed of PP_F32. */
#define PP_MIXED 2

/* status codes */
#define PP_OK 0
#define PP_EINVAL (-1) /* NULL / misaligned pointer, N < 1, delta < 0, non-finite scalar, bad precision/flags */
#define PP_ECUDA (-2)  /* a CUDA runtime call failed (message in pp_last_error) */
#define PP_ENOMEM (-3) /* workspace allocation failed */

/* pp_step_kdk flags */
#define PP_ACC_VALID 1u /* acc already holds a(t0) for the incoming positions: skip the initial gravity solve */

/* pp_configure keys */
#define PP_CFG_SPLIT_J 1 /* 0 = automatic (default); S >= 1 forces the j-range to be split S ways */
#define PP_CFG_GRAPH 2   /* 1 (default) = pp_step_kdk replays its interior steps from a CUDA graph when N <= 65536 */
#define PP_CFG_PROFILE 3 /* 1 = bracket every pair-sweep launch with CUDA events (pp_profile_read); no graph replay */
#define PP_CFG_EQUAL_MASS 4 /* 1 (default) = j-tiles whose bodies all have the same mass take m_j out of the pair loop
                             * (one pipe operation per pair less); 0 = every tile multiplies by m_j per pair */
#define PP_CFG_SHAPE 5   /* kernel shape class of the pair sweep: 0 = chosen by the launch plan (default), 1 = large
                          * (the throughput shape: 1536-1792 i-bodies per CTA, one CTA per SM), 2 = mid (512 i-bodies
                          * per CTA), 3 = small (one i-body per thread).  Any class is correct at any N; the tests use
                          * this to run the edge cases on every shape */

#define PP_CFG_SYMMETRIC 6 /* the pair sweep that evaluates every UNORDERED pair once (Newton's third law: one evaluation
                            * of eq. (2) serves i <- j and j <- i; 7-9 instead of 11-13 FP32-pipe operations per pair
                            * interaction, 9-11.5 instead of 15-18 FP64).  1 (default) = used for full solves (every
                            * precision; not for i-ranges) of N >= 14000 bodies, if its j-side workspace (N^2/(2B) x 16
                            * or 32 B, B = 2048, at most 48 GB; in bands of 16 GB beyond N = 2^21) can be
                            * allocated -- otherwise the one-sided sweep runs; 0 = never; 2 = always (PP_ENOMEM if the
                            * workspace cannot be allocated; PP_CFG_SHAPE = 1 / 2 then pins its 256- / 128-body j-tile
                            * variant, which is otherwise chosen by size: 128 below N = 98304) */

#define PP_CFG_SYM_BAND_ROWS 7 /* test hook: 0 (default) = the symmetric sweep keeps all its j-side rows when they fit 48 GB
                                * and otherwise works through bands of partner offsets of at most 16 GB of rows;
                                * r >= 1 = bands of at most r partner offsets */

/* Version of the library that was loaded (PPGRAV_VERSION). */
int pp_version(void);

/* Message of the last error raised on the calling thread ("" if none). */
const char* pp_last_error(void);

/* Free the cached workspace of `device` (-1: all devices).  Synchronises that device. */
int pp_release(int device);

/* Tuning / test hook, see PP_CFG_*.  Process-wide. */
int pp_configure(int key, int64_t value);

/* Number of CUDA kernels this library has launched since it was loaded (all threads). */
int64_t pp_launch_count(void);

/* With PP_CFG_PROFILE on: waits for the recorded pair-sweep launches and returns out2 (host) =
 * { their summed device time in milliseconds, their number } since the previous read, then forgets them.
 * This is how bench.py obtains the average duration of the dominant kernel without a profiler. */
int pp_profile_read(double* out2);

/* Gravity solve, eq. (1)-(2): the paper's "Gravity Force Computation" kernel.
 *   pos  [N,3] in,  mass [N] in,  acc [N,3] out,  pot [N] out or NULL (skip the potential).
 * O(N^2): N(N-1) ordered pair interactions.  PP_F32: FP32 pair arithmetic, FP32 blocked + compensated sums.
 * PP_F64: FP64 throughout.  acc/pot must not alias pos/mass. */
int pp_forces(const void* pos, const void* mass, void* acc, void* pot, int64_t N, double G, double delta,
              int precision, void* stream);

/* The same gravity solve restricted to the i-bodies [i_begin, i_begin + i_count): every GPU of a multi-GPU run
 * "calculates the dynamics of N/k particles" against all N j-bodies, so
 *   pos [N,3], mass [N] in (all bodies);  acc [i_count,3] out;  pot [i_count] out or NULL.
 * Per body the arithmetic is that of pp_forces.  The launch plan is made for the range (i_count i-bodies against N
 * j-bodies), so it may pick another shape class or split-j factor than the full solve; a row is bit-identical to
 * the corresponding row of pp_forces exactly when both solves use the same j-tile size and the same split-j factor
 * (pp_plan_query; PP_CFG_SHAPE and PP_CFG_SPLIT_J pin them), otherwise equal to summation-order round-off.
 * PP_EINVAL if the range is empty or leaves [0, N). */
int pp_forces_range(const void* pos, const void* mass, void* acc, void* pot, int64_t N, int64_t i_begin,
                    int64_t i_count, double G, double delta, int precision, void* stream);

/* One "Update System" pass on n bodies, for callers that sequence the step themselves (the sharded
 * step in paper_1803_01190_b200/sharded.py):  vel += kick * acc;  then, if dt != 0,  pos += dt * vel.
 * kick = dt/2, dt = dt is the opening half-kick + drift of eqs. (5)-(6); kick = dt/2, dt = 0 is the closing half-kick
 * of eq. (7).  pos, vel [n,3] in/out;  acc [n,3] in. */
int pp_kick_drift(void* pos, void* vel, const void* acc, int64_t n, double kick, double dt, int precision,
                  void* stream);

/* nsteps kick-drift-kick steps of size dt, eqs. (5)-(7), in the algebraically identical
 * half-kick form  v += dt/2 a(t);  r += dt v;  a(t+dt) = forces(r);  v += dt/2 a(t+dt)  -- the paper's "Update
 * System" kernel around one gravity solve per step.
 *   pos, vel [N,3] in/out;  mass [N] in;  acc [N,3] in/out: with PP_ACC_VALID it holds a(t0) on entry (no initial
 *   solve); on return it always holds a(t0 + nsteps*dt), ready to be passed back with PP_ACC_VALID.
 *   pot [N] out or NULL: if given, the LAST gravity solve of the call also produces Phi_i at t0 + nsteps*dt in the
 *   state precision (one more pipe operation per pair in that solve only), ready for pp_invariants; if the call
 *   performs no solve (nsteps == 0 with PP_ACC_VALID) pot is left untouched.
 * nsteps == 0 only (re)computes acc.  Force evaluations performed: nsteps (+1 without PP_ACC_VALID).
 * Kernel launches: 1 (tile masses) + 3 for a cold start + 1 (kick+drift+pack) + 2 per interior step boundary
 * (pair sweep, fused update pass) + 2 (last sweep, finalize+kick) = 2 nsteps + 2 (+3); the symmetric sweep adds one per
 * call (block masses) and, beyond N = 2^21, one sweep and two fold launches per band of partner offsets.  For N <= 65536 the interior
 * steps are replayed from a CUDA graph that is kept while the arguments do not change (also when `stream` is the legacy
 * default stream: the replay then runs on an internal stream, ordered with `stream` by events). */
int pp_step_kdk(void* pos, void* vel, const void* mass, void* acc, void* pot, int64_t N, double dt, int64_t nsteps,
                double G, double delta, int precision, unsigned flags, void* stream);

/* Conserved integrals, eqs. (8)-(10) plus centre of mass (Fig. 6).
 *   out16 (device, 16 doubles) = { E, K, W, Px, Py, Pz, Lx, Ly, Lz, Cx, Cy, Cz, M, 0, 0, 0 }
 *   K = sum m v^2/2;  W = (1/2) sum_i m_i Phi_i  (negative; j != i);  E = K + W;  P = sum m v;  L = sum m r x v.
 * State arrays are `precision`; all sums are accumulated in FP64 with compensation regardless.
 *   pot: Phi_i [N] in the state precision as returned by pp_forces, or NULL -- then an O(N^2) FP64 potential pass
 *   with compensated accumulation is run on the (promoted) state. */
int pp_invariants(const void* pos, const void* vel, const void* mass, const void* pot, int64_t N, double G,
                  double delta, int precision, double* out16, void* stream);

/* pp_invariants for callers that must not allocate (code under CUDA-graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc).  Same kernels, same outputs (bit-identical to pp_invariants with the same `pot`); what differs:
 *   - the kernels' scratch (per-block partial sums, 296 x 32 doubles = 75,776 bytes) is a file-scope static __device__
 *     array inside the library instead of the grow-on-demand workspace: every GPU that loads the library holds those
 *     75,776 bytes until the process exits;
 *   - the call performs no cudaMalloc / cudaFree and calls no allocating routine (one cudaGetSymbolAddress per device
 *     the first time, then two kernel launches);
 *   - `pot` (Phi_i in the state precision, as pp_forces / pp_step_kdk return it) is REQUIRED: the O(N^2) potential pass
 *     of pp_invariants(pot = NULL) needs the allocating workspace -> PP_EINVAL;
 *   - N beyond PP_NOALLOC_MAX_N -> PP_EINVAL with a message that names the limit; G and delta are not needed (they
 *     only enter through the potential);
 *   - every call shares the one scratch array, which keeps the previous call's contents (nothing needs clearing: each
 *     launched block overwrites its slot before the final kernel reads it).  Calls on ONE stream follow each other
 *     safely; calls that overlap on the GPU (several streams without ordering, several host threads) RACE on it.
 *   pos, vel [N,3], mass, pot [N]: device, `precision`;  out16: device, 16 doubles, as pp_invariants. */
#define PP_NOALLOC_MAX_N (1ll << 28)
int pp_invariants_noalloc(const void* pos, const void* vel, const void* mass, const void* pot, int64_t N,
                          int precision, double* out16, void* stream);

/* Face-on surface-density map, the diagnostic of Fig. 7:
 *   sigma [ny*nx] (device, doubles, row-major, overwritten) = (sum of m_i over the bodies with
 *   x0 + ix*cell <= x_i < x0 + (ix+1)*cell and y0 + iy*cell <= y_i < y0 + (iy+1)*cell) / cell^2;  z is ignored and
 *   bodies outside the grid are dropped.  pos [N,3], mass [N] in the state precision; the cell index is
 *   floor((x - x0) * (1/cell)) evaluated in FP64 on the promoted coordinate.  Sums use floating-point atomics, so
 *   this diagnostic (unlike the force path) is reproducible only up to summation order (~1e-16 relative).
 *   PP_EINVAL unless cell > 0, nx, ny >= 1 and nx*ny <= 2^26. */
int pp_surface_density(const void* pos, const void* mass, int64_t N, double x0, double y0, double cell, int nx,
                       int ny, int precision, double* sigma, void* stream);

/* Host-buffer variants: same semantics, HOST pointers, synchronous (copies in, computes, copies out). */
int pp_forces_host(const void* pos, const void* mass, void* acc, void* pot, int64_t N, double G, double delta,
                   int precision, void* stream);
int pp_step_kdk_host(void* pos, void* vel, const void* mass, void* acc, void* pot, int64_t N, double dt,
                     int64_t nsteps, double G, double delta, int precision, unsigned flags, void* stream);
int pp_invariants_host(const void* pos, const void* vel, const void* mass, const void* pot, int64_t N, double G,
                       double delta, int precision, double* out16, void* stream);

/* Launch plan the library would use for a full gravity solve of N bodies (with_pot: the sweep that also produces the
 * potential): out16 (host) =
 *   { [0] i-bodies per CTA, [1] j-bodies per tile, [2] split-j factor S, [3] CTAs launched, [4] CTAs resident per SM,
 *     [5] SM count, [6] pipe operations (FP32- or FP64-pipe instructions per lane) per pair EVALUATION on a j-tile of
 *     mixed masses -- fewer by [12] on a tile whose bodies have a common mass, see pp_equal_mass_tiles --,
 *     [7] MUFU operations per evaluation, [8] shape class (0 large, 1 mid, 2 small, 3 = the symmetric sweep,
 *     PP_CFG_SYMMETRIC), [9] threads per CTA, [10] i-bodies per thread, [11] i-blocks,
 *     [12] ordered pairs (pair interactions) one evaluation serves: 1, or 2 for the symmetric sweep,
 *     [13] symmetric sweep: partner blocks H per block, [14] symmetric sweep: bands the partner blocks are cut into
 *     (1 = all j-side rows are kept at once), [15] bytes of device workspace the solve keeps (packed bodies, partial
 *     sums, j-side rows; at most ~64 GB at any N: the rows are capped at 48 GB, 16 GB per band in a banded solve) }. */
int pp_plan_query(int64_t N, int precision, int with_pot, int64_t* out16);

/* How many j-tiles of a gravity solve of these masses have a common mass (and therefore run the pair loop without
 * the per-pair multiplication by m_j): mass [N] (device, `precision`) in; out2 (host) = { j-tiles swept, j-tiles with
 * a common mass }.  Independent of PP_CFG_EQUAL_MASS.  Synchronous.  bench.py uses it to count the pipe operations
 * per pair that were actually executed. */
int pp_equal_mass_tiles(const void* mass, int64_t N, int precision, int64_t* out2, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* PPGRAV_H_ */
