/*
 * vesnet_farfield.h -- C-ABI boundary of the B200-native far-field module of VesNet
 * (arxiv/paper_2606_25569).  Plain C, no CUDA or torch types in any signature.
 *
 * The module is the one conventional, data-parallel piece VesNet keeps beside its
 * networks: "DirectSingleLayerIntegral(X, f)" (Alg. 4 line 3), the
 * O((MN)^2) direct evaluation of the single-layer integral between vesicles that is
 * "done without any approximation" and dominates the time step.
 * Around it, declared further down: the near-field relation and the masked sum (the paper's
 * actual DirectSingleLayerIntegral), free targets, a fast multipole evaluation of the same
 * sums, the elastic force that produces F, and the equal-arclength redistribution.
 *
 * Mathematics (PAPER.md:129-136 eqs 2.8/2.9, :173 trapezoid rule, :140-144 eq 2.10):
 *
 *   U[v,i,:] = 1/(4 pi mu) * sum_{v' != v} sum_{j<npts}
 *                  ( -log|r| I + r r^T / |r|^2 ) F[v',j,:] W[v',j],   r = X[v,i,:] - X[v',j,:]
 *
 * (the extracted paper text prints "+log|r|" and drops the identity; see DESIGN.md
 * reading A1).  W are the trapezoid arclength weights ds = |dX/dalpha| 2 pi / npts with
 * the derivative taken spectrally.
 *
 * Conventions for every call:
 *  - Arrays are contiguous, row-major, interleaved (x, y): X, F, U are [nves, npts, 2],
 *    W is [nves, npts].  `precision` selects storage AND arithmetic: VN_F32 -> float,
 *    VN_F64 -> double for every array of the call.  mu is a host double.
 *  - "device pointer" = memory of the CURRENT CUDA device, owned by the caller, never
 *    freed or retained by the library.  X, F, U must be aligned to one (x, y) pair
 *    (8 B fp32 / 16 B fp64), W to one element.  Outputs are overwritten and must not
 *    alias inputs.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Device
 *    calls only enqueue work and return; scratch memory is stream-ordered
 *    (cudaMallocAsync / cudaFreeAsync on `stream`), so back-to-back calls on one stream
 *    need no host synchronisation and a sequence of calls can be captured into a CUDA graph
 *    (after one eager call per entry point, which performs the lazy per-device initialisation).
 *  - Errors are return codes only; nothing is printed, thrown or aborted.
 *      VN_ERR_INVALID_ARG  null pointer, nves < 1, npts < 1, nves*npts >= 2^31,
 *                          mu not finite or <= 0, bad enum, misaligned pointer
 *      VN_ERR_UNSUPPORTED  current device is not compute capability 10.x (there is no
 *                          fallback of any kind, by design)
 *      VN_ERR_CUDA         a CUDA runtime call failed (allocation, launch)
 *    Argument checks happen before any CUDA call, so they work without a GPU.
 *  - VN_F32 uses the SFU approximations rcp/lg2 (flush-to-zero): squared distances must be normal
 *    fp32 numbers.  vn_farfield_targets additionally shares one reciprocal between two pairs
 *    (t = rcp(a*b), 1/a = t*b), which is exact only while a*b stays inside the fp32 normal range
 *    (1e-9 < |r| < 1e9 in the caller's units); a tile in which that fails (a target on top of a source,
 *    say) is detected and redone with one reciprocal per pair, so that a bad distance spoils the value of
 *    its own target only.  VN_F64 needs normal doubles whose reciprocal is normal.
 *  - Input values are not validated.  A non-finite value anywhere in X, F or W makes EVERY output of
 *    vn_farfield / vn_farfield_masked / vn_farfield_targets NaN (their integer accumulators cannot carry
 *    NaN/Inf point by point; a free target's own coordinates are not checked); the FMM calls, and vn_farfield
 *    for suspensions of at most 1,024 points (one launch, plain floating-point sums), let it propagate
 *    through their arithmetic: at least every output the value contributes to is non-finite.  Points of DIFFERENT vesicles
 *    are assumed distinct; a coincident cross-vesicle pair gives an unspecified (possibly
 *    non-finite) value at that target only (reading A5).  nves == 1 is valid and yields U == 0.
 */
#ifndef VESNET_FARFIELD_H
#define VESNET_FARFIELD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    VN_OK = 0,
    VN_ERR_INVALID_ARG = 1,
    VN_ERR_UNSUPPORTED = 2,
    VN_ERR_CUDA = 3,
    VN_ERR_TOO_LARGE = 4    /* vn_farfield_noalloc_f32 only: more points than the static scratch holds */
} vn_status;

typedef enum { VN_F32 = 0, VN_F64 = 1 } vn_precision;

/* Far-field single-layer potential at every membrane point, own vesicle excluded
 * (north_star).  All pointers are DEVICE pointers.
 * Steps run on the device: pack g = F*W, pair sum over all other vesicles' points,
 * two-level accumulation, scale by 1/(4 pi mu), store.  U is overwritten.
 * Suspensions of at most 1,024 points take a single-launch kernel without scratch memory
 * (one-directional sums, no atomics); larger ones the symmetric pair kernels. */
vn_status vn_farfield(const void *X, const void *F, const void *W,
                      int64_t nves, int64_t npts, double mu,
                      void *U, vn_precision precision, void *stream);

/* Trapezoid arclength weights W[v,j] = (2 pi / npts) |dX_v/dalpha (alpha_j)|,
 * alpha_j = 2 pi j / npts, derivative by Fourier differentiation with the unmatched
 * k = npts/2 mode dropped for even npts (reading A4).
 * X, W are DEVICE pointers.  W is overwritten. */
vn_status vn_arclength_weights(const void *X, int64_t nves, int64_t npts,
                               void *W, vn_precision precision, void *stream);

/* The whole hot path from HOST buffers: copies X, F (and W when W != NULL) to the
 * device, computes W with vn_arclength_weights when W == NULL, runs vn_farfield and
 * copies U back; returns after U is complete (synchronous).  X, F, W, U are HOST
 * pointers (pinned memory makes the copies asynchronous to the host but is not
 * required).  Device buffers are cached per process and grown on demand. */
vn_status vn_farfield_host(const void *X, const void *F, const void *W,
                           int64_t nves, int64_t npts, double mu,
                           void *U, vn_precision precision);

/* ---- row f-1: the paper's DirectSingleLayerIntegral with its near-field mask ------------------
 *
 * Near-field relation ("A vesicle is considered in the near-field of the point x if
 * the distance of x to the vesicle is less than or equal to the arclength spacing", :248 |d| <= h,
 * :426 Alg. 4 line 4 FindNearFieldPoints):
 *
 *   near(t, v')  <=>  v' != ves(t)  and  min_j |X[t] - X[v',j]| <= h_v',   h_v' = max_j W[v',j]
 *
 * (h = the largest trapezoid weight of the source vesicle, reading N1; the distance to
 * the membrane is the distance to its nearest discretisation point.)  The decision is taken in
 * double arithmetic on the stored values for both precisions.  Output is CSR over the P = nves*npts
 * target points t = v*npts + i, all DEVICE pointers:
 *   near_ptr[P+1]  int64, near_ptr[0] = 0, near_ptr[P] = number of near (point, vesicle) pairs
 *   near_ves[...]  int32, for each t the near vesicles v' in ascending order
 * `capacity` is the number of int32 entries near_ves can hold; entries at positions >= capacity are
 * not written (near_ptr is always complete, so the caller detects overflow by near_ptr[P] >
 * capacity and calls again).  near_ves may be NULL with capacity 0: count only. */
vn_status vn_near_pairs(const void *X, const void *W, int64_t nves, int64_t npts,
                        int64_t *near_ptr, int32_t *near_ves, int64_t capacity,
                        vn_precision precision, void *stream);

/* vn_farfield with the contribution of every near vesicle set to zero ("direct
 * integration with boolean masks to set neighboring vesicles' contribution to zero", :425 Alg. 4
 * line 3):
 *
 *   U[t,:] = 1/(4 pi mu) sum_{v' != ves(t), v' not near t} sum_j K(X[t]-X[v',j]) F[v',j,:] W[v',j]
 *
 * near_ptr / near_ves: the CSR relation as written by vn_near_pairs (DEVICE pointers, complete:
 * near_ptr[P] entries readable in near_ves; near_ves may be NULL only if near_ptr[P] == 0).  Any
 * relation in that format is accepted (v' == ves(t) entries are a caller error, not checked).
 * The near contributions are evaluated in double and leave the accumulators before the final
 * rounding.  Other arguments as vn_farfield. */
vn_status vn_farfield_masked(const void *X, const void *F, const void *W,
                             int64_t nves, int64_t npts, double mu,
                             const int64_t *near_ptr, const int32_t *near_ves,
                             void *U, vn_precision precision, void *stream);

/* ---- row f-4: free targets ------------------------------------------------------------------
 * Velocity induced at nt points Xt[nt,2] that lie on no membrane by ALL vesicles (eq 2.8 summed
 * over every vesicle with the trapezoid rule; the velocity-field
 * evaluation behind the paper's streamline figures):
 *
 *   Ut[q,:] = 1/(4 pi mu) sum_{v'} sum_j K(Xt[q]-X[v',j]) F[v',j,:] W[v',j]
 *
 * No vesicle is excluded; a target closer to a membrane than its point spacing gets the plain
 * trapezoid value (inaccurate there by the nature of the rule).  Xt, Ut: DEVICE
 * pointers, [nt,2] interleaved, pair-aligned; nt == 0 is valid and does nothing.  Ut overwritten. */
vn_status vn_farfield_targets(const void *Xt, int64_t nt,
                              const void *X, const void *F, const void *W,
                              int64_t nves, int64_t npts, double mu,
                              void *Ut, vn_precision precision, void *stream);

/* ---- row f-4, second half: the far-field sum by a fast multipole method -----------------------
 * The same quantity as vn_farfield (own vesicle excluded, same conventions), computed in O(P) by the
 * 2-D fast multipole method the paper points to as future work ("Applying the fast multipole method
 * ... will make it scale as O(M), but an applicable GPU implementation is beyond the scope of this
 * paper"; Greengard & Rokhlin 1987 cited PAPER.md:173).  It is an APPROXIMATION:
 * `order` = p, the number of terms kept in the multipole / local expansions (2 <= p <= 48, or 0 for
 * the default that meets vn_farfield's tolerance: 14 for VN_F32, 38 for VN_F64); the
 * relative L2 truncation error falls like 0.45^p (measured on the synthetic suspensions: p = 12
 * about 3e-6, p = 20 about 5e-9, p = 38 about 1e-13) and the largest point-wise error, relative to the largest
 * velocity, is about 15 times that (targets near the corner of their leaf box): 8e-5 at p = 12, 1.7e-5 at the
 * default p = 14; vn_farfield stays the exact path.  The expansions are formed in the frame of the root square's
 * centre, so the accuracy does not depend on where the suspension sits.
 * The expansions are double for both storage precisions; the direct part over neighbouring leaves runs
 * in the storage precision (VN_F32: the same SFU pair arithmetic as vn_farfield, error about 1e-6).  Uniform quadtree over the bounding square of the points; a strongly
 * non-uniform point distribution costs time (crowded leaves), not accuracy.  Results are bitwise
 * reproducible.  Scratch: about 100 * (p+1) bytes per leaf box plus 120 bytes per point.  Stream-ordered and
 * capturable into a graph like the other calls; two of its kernels hold a grid-wide barrier and are launched with
 * the cooperative attribute (calls in flight on several streams at once are safe).
 * near_ptr / near_ves: NULL for the plain sum (vn_farfield's quantity), or the CSR near-field
 * relation of vn_near_pairs: then the listed vesicles' contributions are zeroed as in
 * vn_farfield_masked (the paper's DirectSingleLayerIntegral in O(P)). */
vn_status vn_farfield_fmm(const void *X, const void *F, const void *W,
                          int64_t nves, int64_t npts, double mu, int order,
                          const int64_t *near_ptr, const int32_t *near_ves,
                          void *U, vn_precision precision, void *stream);

/* vn_farfield_targets (free targets, all vesicles contribute) by the same fast multipole method: the
 * sources build the tree and the local expansions, the nt targets are sorted into the same leaves.
 * Same approximation and `order` semantics as vn_farfield_fmm, same conventions as vn_farfield_targets. */
vn_status vn_farfield_targets_fmm(const void *Xt, int64_t nt,
                                  const void *X, const void *F, const void *W,
                                  int64_t nves, int64_t npts, double mu, int order,
                                  void *Ut, vn_precision precision, void *stream);

/* ---- row f-2: the elastic membrane force (the producer of F) -----------------------------------
 * PAPER.md:123 eq 2.7, :319 Fig. 5b:
 *
 *   F[v,j,:] = -kappa_b X_ssss + (sigma X_s)_s   at point j of vesicle v,
 *   d/ds = |dX/dalpha|^-1 d/dalpha, d/dalpha = Fourier derivative with the unmatched
 *   k = npts/2 mode dropped, the four arclength derivatives applied one after the other without
 *   filtering (readings A4, E1).
 *
 * X[nves,npts,2], sigma[nves,npts] (membrane tension per point), F[nves,npts,2]: DEVICE pointers in
 * the call's precision; kappa_b: host double (bending stiffness, one value for all vesicles, any
 * finite value).  Arithmetic is double inside for both precisions.  npts <= 1024 (one vesicle lives
 * in one block's shared memory), else VN_ERR_INVALID_ARG.  F is overwritten and must not alias
 * the inputs.  The result is conditioned like a fourth derivative: rounding of X is amplified by
 * about (npts/2)^4 / |dX/dalpha|^4. */
vn_status vn_elastic_force(const void *X, const void *sigma, int64_t nves, int64_t npts,
                           double kappa_b, void *F, vn_precision precision, void *stream);

/* ---- row f-3: redistributing points equally in arclength ----------------------------------------
 * PAPER.md:331-335 (sec 4.2), called three times per time step.  Per vesicle:
 *   1. trigonometric interpolation of X to M = 6 npts nodes ("upsample by a factor of 6");
 *   2. arclength l_m at those nodes: |dX/dalpha| by Fourier differentiation, integrated through the
 *      Fourier series of |dX/dalpha| on the fine grid; L = l_M the total length;
 *   3. for k = 0 .. npts-1: target arclength k L / npts, located in the increasing sequence l_0..l_M,
 *      Xnew[v,k,:] = linear interpolation of the two upsampled points that bracket it.
 * (readings R1-R5 state what the paper leaves open: Nyquist handling, spectral
 * integration, point 0 stays in place, positions interpolated with the same weight as arclength.)
 * The new points are equispaced in arclength up to the piecewise-linear error of step 3
 * (relative spacing error about 1e-4 at npts = 128) and lie on the chords of the upsampled
 * polygon.  X, Xnew: DEVICE pointers, [nves,npts,2] in the call's precision (arithmetic is double
 * inside); Xnew is overwritten and must not alias X.  3 <= npts <= 512, else VN_ERR_INVALID_ARG.
 * The arclength sequence is assumed increasing (true whenever the curve is resolved). */
vn_status vn_redistribute_arclength(const void *X, int64_t nves, int64_t npts, void *Xnew,
                                    vn_precision precision, void *stream);

/* Profiling aid (bench.py's roofline figure): while enabled, every vn_farfield /
 * vn_farfield_host / vn_farfield_masked / vn_farfield_targets call records a CUDA event pair on its
 * stream around the pair kernel alone (not the pack / finish / correction kernels).  vn_profile_read waits for the recorded events,
 * writes up to max_entries durations in milliseconds (oldest first) into the HOST array
 * ms, forgets them, and returns how many it wrote (or -1 on a CUDA error).  vn_profile_enable(0) also destroys
 * whatever events were recorded and not read. */
vn_status vn_profile_enable(int enable);
int64_t vn_profile_read(double *ms, int64_t max_entries);

/* One suspension on several GPUs.  The pair kernel evaluates every
 * unordered pair of points once and scatters into both points' accumulators, so the work is dealt out by BLOCKS of
 * the pair walk, not by targets: with all sources known to every device (one all-gather of X, F, W), device `part`
 * of `nparts` runs vn_farfield_partial, which executes blocks part, part + nparts, ... of the same grid vn_farfield
 * would run and leaves the RAW fixed-point accumulators in acc: 2 (VN_F32) or 4 (VN_F64) 64-bit integer words per
 * point, [nves*npts*2] or [nves*npts*4] int64, overwritten.  Integer addition is associative, so summing the
 * parts' accumulators word by word in any order (one integer reduce-scatter over the devices, 16 / 32 bytes per
 * point) gives bit for bit the accumulators of the single-device call.  vn_farfield_finish then turns any
 * contiguous range of `count` points of summed accumulators (pointer to the first word of the range) into
 * velocities U[count,2]: scale by 1/(4 pi mu), round once.  gmax (8 bytes, 8-byte aligned, written by
 * vn_farfield_partial, identical on every device because every device packs all sources) carries the scale of
 * the fixed-point format; npoints_total = nves*npts of the whole suspension.  part = 0, nparts = 1 followed by
 * vn_farfield_finish over all points IS vn_farfield.  All pointers are DEVICE pointers; asynchronous on `stream`.
 * VN_ERR_INVALID_ARG additionally for part < 0, nparts < 1, part >= nparts, count < 0. */
vn_status vn_farfield_partial(const void *X, const void *F, const void *W, int64_t nves, int64_t npts,
                              int32_t part, int32_t nparts, void *acc, void *gmax,
                              vn_precision precision, void *stream);
vn_status vn_farfield_finish(const void *acc, const void *gmax, int64_t npoints_total, int64_t count, double mu,
                             void *U, vn_precision precision, void *stream);

/* Self-check of the pair kernels' shared-memory ring (stands in for compute-sanitizer's
 * racecheck / initcheck, which cannot be run on the development pool).  Computes what vn_farfield computes, always
 * with the symmetric pair kernels (whatever the size), in a verification build of them: every source record a warp
 * reads from a ring stage is compared, bit for bit, with its original in global memory, so a stage refilled by the
 * bulk copy while a warp still reads it, or read before its copy has landed, is counted; and the scratch memory is
 * filled with 0xFF bytes before use, so a read of scratch that no kernel wrote shows in U.  Synchronous: waits for
 * `stream`, then writes the number of mismatching record reads into the HOST variable *mismatches (0 = clean).
 * U (DEVICE, overwritten) must equal vn_farfield's U bit for bit when the suspension has more than 1,024 points. */
vn_status vn_selfcheck(const void *X, const void *F, const void *W, int64_t nves, int64_t npts, double mu,
                       void *U, vn_precision precision, void *stream, int64_t *mismatches /* HOST */);

/* Measured issue rates of the arithmetic pipes that bound the pair kernels (the nominal
 * lane counts "must be confirmed by microbenchmark").  Runs six register-only stream
 * kernels of this library on `stream` (about 60 ms in all), waits for them, and writes into the HOST array
 * rates[8]: lane-operations per second of [0] packed FFMA2 (fma.rn.f32x2, counted as two per thread),
 * [1] FFMA, [2] MUFU (rcp.approx and lg2.approx, half each), [3] DFMA; [4] the device's SM count; [5], [6] FFMA2
 * and DFMA streams whose three operands are different registers in every instruction (no operand reuse between
 * neighbours: what the register file feeds the pipes when all inputs change); [7] zero (reserved).
 * The best of three launch shapes (16 / 32 / 64 warps per SM, eight independent chains per thread) is reported.
 * Synchronous; not capturable into a graph.  bench.py calls it once per run for roofline.peak_measured. */
vn_status vn_pipe_peaks(double *rates /* HOST, 8 entries */, void *stream);

/* vn_farfield without any allocation, single precision (the same sum, the same kernels).
 * For callers that cannot call cudaMalloc: code under CUDA graph / stream capture, tight serving loops, harnesses
 * that forbid it.  vn_farfield takes 48 bytes of scratch per point from the stream-ordered allocator for every call
 * above 1,024 points; this entry point keeps that scratch in a static device array of the library instead and calls
 * no cudaMalloc*, cudaFree* or allocating library routine (with vn_profile_enable off).  The price is a LIMIT and a
 * standing cost: at most vn_noalloc_max_points() = 262,144 points (nves*npts; BASELINE.json configs[0..3]), and the
 * array -- 12 MiB + 256 B -- is held by every GPU that loads the library until the process exits.
 * X, F [nves,npts,2], W [nves,npts], U [nves,npts,2]: float, DEVICE pointers, the caller's; U is overwritten and
 * must not alias an input.  Always the symmetric pair kernel (also below 1,024 points), with the grid vn_farfield
 * uses: above 1,024 points U equals vn_farfield's bit for bit.  Asynchronous on `stream`.
 * Returns VN_ERR_TOO_LARGE for nves*npts > vn_noalloc_max_points() (checked before any CUDA call, nothing is
 * launched), otherwise vn_farfield's codes.  All calls on a device SHARE the array, which keeps the previous call's
 * contents (the call clears what must start at zero): calls on one stream are ordered and safe; calls whose
 * kernels overlap on the GPU -- two streams, two graphs replayed concurrently, two host threads on two streams --
 * race on it and give undefined results.  The first call on a device looks the array's address up
 * (cudaGetSymbolAddress, device current) and queries the kernel's occupancy: make it outside a capture. */
vn_status vn_farfield_noalloc_f32(const void *X, const void *F, const void *W, int64_t nves, int64_t npts,
                                  double mu, void *U, void *stream);
int64_t vn_noalloc_max_points(void);

/* Host-only introspection (no CUDA call, works without a GPU): the work decomposition vn_farfield would use
 * for nves x npts points when `resident_blocks` blocks of the pair kernel fit on the device at once
 * (148 SMs x 3 on a B200).  plan[0] = points per super-tile (target block), plan[1] = source tiles per
 * super-tile, plan[2] = number of super-tiles n_st, plan[3] = chunks per super-tile (grid = n_st * chunks),
 * plan[4] = points per source tile.  Block (I, c) walks chunk c of the list  { tiles of I itself; tiles of
 * super-tiles I+1 .. I+S_I (mod n_st) },  S_I = floor((n_st-1)/2) (+1 for I < n_st/2 when n_st is even), which
 * visits every unordered pair of super-tiles exactly once.  Used by the CPU tests of the host logic. */
vn_status vn_plan_farfield(int64_t nves, int64_t npts, vn_precision precision, int32_t resident_blocks,
                           int32_t *plan /* HOST, 5 entries */);

/* Number of kernels of this library launched by the calling process so far
 * (all entry points, all streams).  Used by bench.py to report gpu_launches. */
int64_t vn_launch_count(void);

/* Static, NUL-terminated description of a status code. */
const char *vn_status_string(vn_status s);

/* Library version: major*10000 + minor*100 + patch (this header: 0.2.1 = 201). */
#define VN_VERSION 201
int vn_version(void);

#ifdef __cplusplus
}
#endif

#endif /* VESNET_FARFIELD_H */
