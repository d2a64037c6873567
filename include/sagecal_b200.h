/*
 * sagecal_b200.h -- C ABI of libsagecal_b200.so
 *
 * The data-parallel hot path of SAGECal direction-dependent calibration
 * (arXiv 1910.13908; the problem statement is BASELINE.json:5 "north_star",
 * the paper itself, only says "a single calibration solution will
 * be derived for each cluster") as hand-written CUDA for one NVIDIA B200
 * (sm_100a).  Readings of everything the paper leaves open: DESIGN.md §3.
 *
 * Conventions
 *   N stations, B = N(N-1)/2 baselines (p<q, no autocorrelations), T time
 *   slots, F channels, K clusters.  rows = T*B, samples = rows*F.
 *   Canonical row order: row r = t*B + b, b(p,q) = p*N - p(p+1)/2 + (q-p-1).
 *   Complex numbers are interleaved {re, im} doubles (sagecal_c128, bit
 *   compatible with cuDoubleComplex / torch.complex128 / C99 double complex).
 *   A 2x2 matrix is row-major [XX, XY, YX, YY].
 *   Visibilities, residuals:  [rows][F][4] c128 (64 B per sample).
 *   Coherencies of K clusters, chosen by `coh_format`:
 *     SAGECAL_COH_FULL   [K][rows][F][4] c128  (general 2x2, 64 B/sample)
 *     SAGECAL_COH_SCALAR [K][rows][F]    c128  (C = c*I2, exact when every
 *                         source has Q=U=V=0; 16 B/sample)
 *   Jones matrices: [K][N][4] c128.
 *
 * Pointers
 *   "dev"  = device pointer owned by the caller (e.g. a torch tensor); must be
 *            32-byte aligned (torch allocations are 512-byte aligned).
 *   "host" = host pointer, read during the call (small descriptors only),
 *            may be freed on return.
 *   The library never allocates caller-visible memory: scratch comes from the
 *   caller's `workspace` (dev, 256-byte aligned), sized by
 *   sagecal_workspace_bytes().  `stream` is a cudaStream_t (NULL = default
 *   stream).  Every call is asynchronous on `stream` and never synchronises
 *   the device; scalar results are device pointers.
 *
 * Errors
 *   Every function returns 0 on success or a negative SAGECAL_E* code; nothing
 *   is enqueued when argument validation fails.  No exceptions, no aborts.
 */
#ifndef SAGECAL_B200_H
#define SAGECAL_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { double re, im; } sagecal_c128;

#define SAGECAL_OK            0
#define SAGECAL_EINVAL       (-1)  /* bad shape, NULL pointer, misaligned pointer, bad enum */
#define SAGECAL_EWORKSPACE   (-2)  /* workspace NULL or smaller than sagecal_workspace_bytes() */
#define SAGECAL_ECUDA        (-3)  /* a CUDA call failed: see sagecal_last_cuda_error() */
#define SAGECAL_EUNSUPPORTED (-4)  /* valid request this build does not implement */
#define SAGECAL_ESTATICLIMIT (-5)  /* request exceeds the fixed device scratch of a no-allocation entry point */

#define SAGECAL_COH_FULL   0
#define SAGECAL_COH_SCALAR 1

/* `lm_mode` of sagecal_sage_calibrate: how the n_lm+1 cost/gradient/J^H J evaluations of an M-step are computed.
 * Both follow the same LM trajectory and agree to rounding. */
#define SAGECAL_LM_COMPRESSED 0  /* default: per-baseline time/frequency statistics of the residual, taken once per
                                    (EM iteration, cluster) in the same streaming kernel that writes back the previous
                                    clusters; the n_lm+1 evaluations and the LM control then run in one cooperative
                                    kernel that reads 392 B per baseline instead of 128 B per sample */
#define SAGECAL_LM_DIRECT     1  /* every evaluation streams the cluster's T*F samples (sagecal_lm_cost_grad_jtj) */
#define SAGECAL_LM_FULLGN     2  /* the other reading of "per-station-block J^H J ... small dense per-cluster solve"
                                    (DESIGN.md §3 Q1, §5.6): the FULL 8N x 8N Gauss-Newton matrix, one off-diagonal 8x8
                                    block per baseline, damped Cholesky with cuSOLVER, on the compressed statistics.
                                    A different iteration (it converges in a handful of steps), not the hot path;
                                    needs the SAGECAL_WS_CALIBRATE_FULLGN workspace (3 x (8N)^2 doubles more). */
#define SAGECAL_LM_PERCLUSTER 3  /* SAGECAL_LM_COMPRESSED with the cluster-by-cluster streaming kernel forced on (one
                                    read and one write of R per cluster, wbstat.cu).  SAGECAL_LM_COMPRESSED itself works
                                    on groups of 4 consecutive clusters whenever an M-step is a single chunk
                                    (n_lm <= SAGECAL_LM_RECENTRE): one read and one write of R per group, statistics
                                    corrected inside a group through cross grams of the coherencies, on the FP64 tensor
                                    cores for 2x2 coherencies (DESIGN.md §5.5 "cluster groups"); longer M-steps take the
                                    cluster-by-cluster route.  Same trajectory to rounding either way. */
/* compressed mode re-takes the statistics at the accepted Jones every this many trial steps of one M-step */
#define SAGECAL_LM_RECENTRE  10

/* `what` of sagecal_workspace_bytes */
#define SAGECAL_WS_LM_PASS   1          /* sagecal_lm_cost_grad_jtj: per-unit partial sums and per-baseline records */
#define SAGECAL_WS_CALIBRATE 2          /* sagecal_sage_calibrate, lm_mode COMPRESSED or DIRECT, either coherency format:
                                           the above + per baseline K x 16 + 5 x 34 doubles of statistics and 6 x 32 doubles of
                                           cross grams per group of 4 clusters (3.7 GB at N=512, K=50) */
#define SAGECAL_WS_CALIBRATE_FULLGN 3   /* lm_mode FULLGN: the above + 3 x (8N)^2 + 58 x B doubles (0.47 GB more at N=512) */

/* Speed of light used to turn uvw in metres into wavelengths (m/s). */
#define SAGECAL_C0 299792458.0

const char* sagecal_strerror(int code);
/* cudaError_t of the last failing CUDA call made by this library on this host thread (0 = none). */
int sagecal_last_cuda_error(void);
/* "major.minor.patch" of the library. */
const char* sagecal_version(void);

/* Bytes of device scratch the call named by `what` needs for this shape (0 if none).
 * Returns 0 for invalid arguments as well; the call itself then reports SAGECAL_EINVAL. */
size_t sagecal_workspace_bytes(int what, int nstations, int ntime, int nchan, int nclus);

/*
 * Coherency prediction (BASELINE.json:5 "The first is per-cluster model prediction";
 * SURVEY.md §8(a) rows 8a-0, 8a-1; DESIGN.md §3 readings Q2, Q4, Q5):
 *
 *   C_k[r][c] = sum_{s in cluster k} B_s(f_c) * exp(-2 pi i (f_c/c0) (u_r l_s + v_r m_s + w_r (n_s - 1)))
 *   B_s(f)    = (f/f0)^alpha_s * [[I+Q, U+iV], [U-iV, I-Q]],     n_s - 1 = -(l^2+m^2)/(1+sqrt(1-l^2-m^2))
 *
 * nstations, ntime : N, T; rows = T*N(N-1)/2 (N >= 2, T >= 1).
 * freqs_host [F]   : channel frequencies in Hz (host), F >= 1.  Uniformly spaced
 *                    channels use a per-channel phasor recurrence; anything else one sincos per channel.
 * f0               : reference frequency of the flux law, Hz (> 0).
 * uvw              : dev [rows][3] f64, metres, for the baseline as ordered (p, q).
 * nclus, cluster_offset_host [K+1] : sources of cluster k are [offset[k], offset[k+1]) (host, non-decreasing,
 *                    offset[0] = 0).  An empty cluster yields zeros.
 * src_l, src_m, src_I, src_alpha : dev [S_tot] f64.  src_Q/U/V : dev [S_tot] or all three NULL = unpolarised.
 * coh_format       : SAGECAL_COH_FULL, or SAGECAL_COH_SCALAR (then Q/U/V must be NULL).
 * coh              : dev out, layout per coh_format.
 * precision        : 0 = float64 throughout (parity 1e-10); 1 = mixed: float64 phase and range reduction,
 *                    float32 sincos polynomial and flux product, float64 accumulation (parity 1e-5).
 * workspace        : dev scratch >= sagecal_predict_workspace_bytes(F, S_tot) (the prepared source table).
 * Limits: F <= 512, K <= 1024 (descriptors travel as kernel parameters, so the call needs no host->device copy).
 */
size_t sagecal_predict_workspace_bytes(int nchan, int nsrc_total);
/* The workspace that lets unpolarised float64 predictions run in station form (below): the size above plus room for the
 * station phasors of as many time slots as fit 2 GiB (at least one; the slots are then predicted in chunks).  With
 * the smaller workspace the call still works and predicts per baseline. */
size_t sagecal_predict_workspace_bytes_station(int nstations, int ntime, int nchan, int nclus, int nsrc_total);
/* How unpolarised float64 predictions are computed (process-wide):
 *   0 (default): in STATION form on the FP64 tensor cores whenever the uvw are differences of station coordinates
 *      (u_pq = u_0q - u_0p to rounding, checked on the device in the same call: true for any interferometer) and the
 *      workspace has room for one time slot's station phasors (sagecal_predict_workspace_bytes_station), else as
 *      below;
 *   1: always one phasor per (baseline, source).
 * Both agree with the definition above to the parity bound.  Returns SAGECAL_EINVAL for any other value. */
int sagecal_predict_set_form(int form);
int sagecal_predict_coherencies(
    int nstations, int ntime, int nchan,
    const double* freqs_host, double f0,
    const double* uvw,
    int nclus, const int* cluster_offset_host,
    const double* src_l, const double* src_m,
    const double* src_I, const double* src_Q, const double* src_U, const double* src_V,
    const double* src_alpha,
    int coh_format, sagecal_c128* coh, int precision,
    void* workspace, size_t workspace_bytes, void* stream);

/*
 * sagecal_predict_coherencies for callers that cannot allocate device memory (code under CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc): same arguments without the workspace, same kernels, same result bit for
 * bit.  The prepared source table lives in a fixed device array of SAGECAL_PREDICT_STATIC_BYTES that every GPU which
 * loads the library holds until the process exits; the call allocates and frees nothing (no cudaMalloc / cudaFree, no
 * allocating library routine) and makes no host<->device copy.
 * Limit: sagecal_predict_workspace_bytes(nchan, S_tot) <= sagecal_predict_static_bytes() (2 MiB: e.g. 7 900 sources
 * x 8 channels, almost 4 times configs[4]'s sky model); beyond it the call returns SAGECAL_ESTATICLIMIT and launches nothing.
 * All calls on a device share the one array, which keeps the previous call's table; every call rewrites the part it
 * reads, so nothing needs clearing.  Calls that may overlap on the GPU (different streams, or two host threads) RACE
 * on it: serialise them on one stream, or use sagecal_predict_coherencies with a workspace per stream.
 */
#define SAGECAL_PREDICT_STATIC_BYTES (2 * 1024 * 1024)
size_t sagecal_predict_static_bytes(void);
int sagecal_predict_coherencies_static(
    int nstations, int ntime, int nchan,
    const double* freqs_host, double f0,
    const double* uvw,
    int nclus, const int* cluster_offset_host,
    const double* src_l, const double* src_m,
    const double* src_I, const double* src_Q, const double* src_U, const double* src_V,
    const double* src_alpha,
    int coh_format, sagecal_c128* coh, int precision,
    void* stream);

/*
 * Prediction fused with the initial residual (rows 8a-0 .. 8a-2 of SURVEY.md §8(a) in one pass; BASELINE.json:5 "the
 * Jones-corrupted residual V_pq - J_p C_pq J_q^H ... with the other clusters' J_p C J_q^H subtracted"):
 *
 *   coh[k]   = sagecal_predict_coherencies' C_k for every cluster (same arithmetic, float64, bit-identical)
 *   residual = vis - sum_k J_{k,p} C_k J_{k,q}^H                      (clusters subtracted in index order)
 *
 * One CTA predicts ALL clusters of its 128 rows and carries the rows' residual in shared memory, so the K
 * coherencies are not read back for the initial residual (69.7 GB at configs[4]).  Follow with
 * sagecal_sage_calibrate(vis = NULL): it then starts from this residual.
 * Arguments as sagecal_predict_coherencies (precision is float64), plus
 * jones    : dev [K][N][4] start Jones (read only).   vis : dev [rows][F][4] (read only).
 * residual : dev out [rows][F][4]; must not alias vis.
 * Errors as sagecal_predict_coherencies; SAGECAL_EINVAL also for nclus < 1 or a NULL / misaligned jones, vis, residual.
 */
int sagecal_predict_residual(
    int nstations, int ntime, int nchan,
    const double* freqs_host, double f0,
    const double* uvw,
    int nclus, const int* cluster_offset_host,
    const double* src_l, const double* src_m,
    const double* src_I, const double* src_Q, const double* src_U, const double* src_V,
    const double* src_alpha,
    int coh_format, sagecal_c128* coh,
    const sagecal_c128* jones, const sagecal_c128* vis, sagecal_c128* residual,
    void* workspace, size_t workspace_bytes, void* stream);

/*
 * Jones corruption and subtraction (BASELINE.json:5 "the Jones-corrupted residual V_pq - J_p C_pq J_q^H";
 * SURVEY.md §8(a) rows 8a-2, 8a-3, 8a-6):
 *
 *   vis_out = vis_in + sign * sum_{k : mask[k]} J_{p,k} C_k J_{q,k}^H        (clusters added in index order)
 *
 * coh              : dev, all K clusters, layout per coh_format.
 * jones            : dev [K][N][4].
 * cluster_mask_host: host [K] bytes, non-zero = include; NULL = all clusters.
 * sign             : -1 subtracts the corrupted model (residual), +1 adds it (simulate / E-step add-back).
 * vis_in, vis_out  : dev [rows][F][4]; vis_out may alias vis_in exactly (in place), no partial overlap.
 *                    vis_in may be NULL = zeros (pure model).
 */
int sagecal_corrupt_subtract(
    int nstations, int ntime, int nchan, int nclus,
    int coh_format, const sagecal_c128* coh, const sagecal_c128* jones,
    const uint8_t* cluster_mask_host, double sign,
    const sagecal_c128* vis_in, sagecal_c128* vis_out, void* stream);

/*
 * One fused Levenberg-Marquardt evaluation pass for ONE cluster (BASELINE.json:5 "the cost, and the gradient
 * and per-station-block J^H J accumulation over all N(N-1)/2 baselines"):
 *
 *   E = x - J_p C J_q^H,   T1 = J_p C,   A = C J_q^H          per sample on baseline (p, q)
 *   cost    = sum ||E||_F^2
 *   grad[p] = sum_{q>p} E A^H  + sum_{q<p} E_{qp}^H T1_{qp}     (d cost = -2 Re sum_p tr(grad[p]^H dJ_p))
 *   jtj[p]  = sum_{q>p} A A^H  + sum_{q<p} T1_{qp}^H T1_{qp}     (2x2 Hermitian PSD; the (p,p) diagonal 8x8 real
 *                                                                block of J^T J acts on a perturbation D as D*jtj[p])
 *
 * x      : dev [rows][F][4]: data with the other clusters' models subtracted.
 * coh_k  : dev, this cluster's coherencies ([rows][F][4] or [rows][F]).
 * jones_k: dev [N][4].
 * cost   : dev out [1] f64.   grad, jtj : dev out [N][4] c128.
 * Sums are formed without global atomics in a fixed order: results are bit-reproducible run to run.  (2x2 coherencies:
 * on the FP64 tensor cores, one warp per baseline; an integer ticket counter decides which block adds the per-station
 * cost partials last -- control flow only, the order of every floating-point sum is fixed.)
 */
int sagecal_lm_cost_grad_jtj(
    int nstations, int ntime, int nchan,
    const sagecal_c128* x, int coh_format, const sagecal_c128* coh_k,
    const sagecal_c128* jones_k,
    double* cost, sagecal_c128* grad, sagecal_c128* jtj,
    void* workspace, size_t workspace_bytes, void* stream);

/*
 * SAGE expectation-maximisation over K clusters with a block-diagonal Levenberg-Marquardt M-step kept entirely on
 * the device (BASELINE.json:5 "the SAGE-EM / Levenberg-Marquardt inner loop run per cluster against the residual
 * with the other clusters' J_p C J_q^H subtracted", item (e)):
 *
 *   R = vis - sum_k J_k C_k J_k^H
 *   for em < n_em, for k < K:   x_k = R + J_k C_k J_k^H
 *       mu = tau * max_p max(M_p[0][0], M_p[1][1]),  nu = 2
 *       n_lm times: dJ_p = G_p (M_p + mu I)^-1;  J' = J + dJ;  rho = (phi(J) - phi(J')) / sum_p [Re tr(G_p^H dJ_p) + mu ||dJ_p||^2]
 *                   accept iff rho > 0 (all finite): J = J', mu *= max(1/3, 1-(2 rho-1)^3), nu = 2;  else mu *= nu, nu *= 2
 *       R = x_k - J_k C_k J_k^H
 *
 * vis     : dev [rows][F][4] (read only), or NULL: `residual` then already holds V - sum_k J_k C_k J_k^H at the start
 *           Jones (written by sagecal_predict_residual) and the initial pass over the coherencies is skipped.
 * coh     : dev, K clusters.
 * jones   : dev [K][N][4], in = start values, out = solution.
 * residual: dev out (in/out with vis == NULL) [rows][F][4]; must not alias vis.
 * tau     : initial damping factor (1e-3 in all configs).
 * lm_mode : SAGECAL_LM_COMPRESSED, SAGECAL_LM_DIRECT, SAGECAL_LM_FULLGN or SAGECAL_LM_PERCLUSTER (above).
 * cost_per_cluster : dev out [K] f64: phi_k at the end of cluster k's last M-step.
 * cost_trace       : dev out [n_em*K + 1] f64 or NULL: ||R||^2 at the start and after every M-step.
 * workspace: dev scratch >= sagecal_workspace_bytes(SAGECAL_WS_CALIBRATE or ..._FULLGN, N, T, F, K).
 * No device->host transfer or synchronisation happens inside the call.  (SAGECAL_LM_FULLGN additionally takes
 * cuSOLVER's own scratch from cudaMallocAsync on `stream`: its size is only known with a device.)
 */
int sagecal_sage_calibrate(
    int nstations, int ntime, int nchan, int nclus,
    const sagecal_c128* vis, int coh_format, const sagecal_c128* coh,
    sagecal_c128* jones, sagecal_c128* residual,
    int n_em, int n_lm, double tau, int lm_mode,
    double* cost_per_cluster, double* cost_trace,
    void* workspace, size_t workspace_bytes, void* stream);

/*
 * Whole-interval convenience entry with HOST buffers (used for end-to-end timing): copies uvw, the source table,
 * the visibilities and the start Jones to the device, runs predict + calibrate, copies Jones, residual and costs
 * back.  Works in an arena of device memory the library allocates (cudaMalloc) on the first call and keeps, per (host
 * thread, device), for the following ones (about 70 GB at configs[4]; grown when a larger interval arrives, handed back
 * by sagecal_host_trim; no memory pool of the device is touched).
 * The visibilities travel on an internal copy stream while the coherencies are predicted, and the last write-back runs
 * in ranges of time slots whose copies to the host overlap the next range's kernel.  Synchronises `stream` and the
 * copy stream before returning.  All array pointers are host pointers (pinned memory recommended: pageable memory
 * serialises the copies).  residual_host / cost_trace_host may be NULL (not copied back).
 */
int sagecal_calibrate_interval_host(
    int nstations, int ntime, int nchan,
    const double* freqs_host, double f0, const double* uvw_host,
    int nclus, const int* cluster_offset_host,
    const double* src_l, const double* src_m, const double* src_I,
    const double* src_Q, const double* src_U, const double* src_V, const double* src_alpha,
    int coh_format,
    const sagecal_c128* vis_host, sagecal_c128* jones_host, sagecal_c128* residual_host,
    int n_em, int n_lm, double tau, int lm_mode,
    double* cost_per_cluster_host, double* cost_trace_host, void* stream);

/*
 * The same, ASYNCHRONOUS: returns once the interval is enqueued, so that a stream of intervals overlaps the
 * device-to-host traffic of one interval (the residual: 25 ms at configs[4], more than any kernel can hide inside its own
 * interval) with the prediction of the next.  Consecutive intervals alternate between TWO arenas (140 GB at configs[4]); the call
 * blocks until the interval before the previous one has finished, so never more than two are in flight per (host
 * thread, device).  The host buffers of an interval -- inputs AND outputs -- belong to the library until
 * sagecal_host_sync returns, or until the call after the next has returned; jones_host is both, so a caller that
 * refills it before every call rotates THREE sets (when call i is made, interval i-3 is home, interval i-2 maybe not).
 * sagecal_host_sync(stream): waits for everything the asynchronous entry enqueued from this host thread on `stream` and
 * on the library's copy streams.  Returns 0 or SAGECAL_ECUDA.
 */
int sagecal_calibrate_interval_host_async(
    int nstations, int ntime, int nchan,
    const double* freqs_host, double f0, const double* uvw_host,
    int nclus, const int* cluster_offset_host,
    const double* src_l, const double* src_m, const double* src_I,
    const double* src_Q, const double* src_U, const double* src_V, const double* src_alpha,
    int coh_format,
    const sagecal_c128* vis_host, sagecal_c128* jones_host, sagecal_c128* residual_host,
    int n_em, int n_lm, double tau, int lm_mode,
    double* cost_per_cluster_host, double* cost_trace_host, void* stream);
int sagecal_host_sync(void* stream);
/* sagecal_host_sync, then hands the arenas the host entries keep cached (one or two, about 70 GB each at configs[4])
 * back to the device.  The next host-entry call allocates again. */
int sagecal_host_trim(void* stream);

/*
 * Measurement-set rows <-> canonical layout, and flags (SURVEY.md §8(f) NEXT-4 "per-row station index arrays
 * (non-canonical order, flags)").  The entry points above address a sample by arithmetic on
 * (time slot, p, q, channel) and carry no mask.  A general row list -- any order, either station orientation, absent
 * (time slot, baseline) pairs, per-sample flags -- is brought into that layout once per interval:
 *
 *   sagecal_rows_to_canonical : row r = (ant1, ant2, tslot) goes to slot tslot*B + b(min, max).  A row with
 *       ant1 > ant2 is the Hermitian transpose of the (min, max) measurement (BASELINE.json:5 "V_qp = V_pq^H"): its
 *       2x2 samples are conjugate-transposed and its uvw negated.  Flagged samples and slots no row maps to come
 *       out as ZERO visibilities with flag 1 (uvw of an empty slot: 0).  Dropped rows: auto-correlations
 *       (ant1 == ant2), indices out of range, and all but the highest-indexed of several rows on one slot.
 *   sagecal_apply_flags       : zeroes the flagged samples of every cluster's coherencies (and of `vis` if not
 *       NULL).  After it E = 0 - J*0*J^H = 0 at flagged samples, so they add nothing to the cost, the gradient,
 *       J^H J or the compressed statistics in ANY entry point above, and their residual is 0 -- at no cost to
 *       the hot loops.  Call it after sagecal_predict_coherencies (which is given the canonical uvw).
 *   sagecal_canonical_to_rows : vis_out[r] = the canonical array's slot of row r, conjugate-transposed back if
 *       ant1 > ant2; dropped rows (row_map < 0) are left untouched.
 *
 * nrows_in             : number of rows in the list (>= 0).
 * ant1, ant2, tslot    : dev [nrows_in] int32.      uvw_in : dev [nrows_in][3] f64, metres, baseline (ant1, ant2).
 * vis_in               : dev [nrows_in][F][4].      flag_in: dev [nrows_in][F] bytes (non-zero = excluded) or NULL.
 * uvw, vis, flags      : dev out, canonical: [T*B][3] f64, [T*B][F][4] c128, [T*B][F] bytes (0/1).
 * row_map              : dev out [nrows_in] int64: 2*slot + (ant1 > ant2), or -1 for a dropped row.
 * status               : dev out [4] int32: {auto-correlations, out-of-range rows, duplicates dropped, empty slots}.
 * workspace            : dev scratch >= sagecal_rows_workspace_bytes(N, T) (one int64 per slot).
 * Integer atomics (slot ownership, counters) are used; the outcome does not depend on their order.
 */
size_t sagecal_rows_workspace_bytes(int nstations, int ntime);
int sagecal_rows_to_canonical(
    int nstations, int ntime, int nchan, int64_t nrows_in,
    const int32_t* ant1, const int32_t* ant2, const int32_t* tslot,
    const double* uvw_in, const sagecal_c128* vis_in, const uint8_t* flag_in,
    double* uvw, sagecal_c128* vis, uint8_t* flags, int64_t* row_map, int32_t* status,
    void* workspace, size_t workspace_bytes, void* stream);
int sagecal_canonical_to_rows(
    int nstations, int ntime, int nchan, int64_t nrows_in, const int64_t* row_map,
    const sagecal_c128* vis_canonical, sagecal_c128* vis_out, void* stream);
int sagecal_apply_flags(
    int nstations, int ntime, int nchan, int nclus, const uint8_t* flags,
    int coh_format, sagecal_c128* coh, sagecal_c128* vis, void* stream);

/*
 * Measurement plumbing (no effect on results).  Every kernel the library launches is counted by kind;
 * kinds are 0..sagecal_kernel_kinds()-1, named by sagecal_kernel_kind_name() ("predict", "corrupt", "lm_pass", ...).
 * sagecal_launch_count : kernels launched by this process since the library was loaded (all kinds).
 * sagecal_profile_enable(mask): from now on bracket every launch whose kind bit is set in `mask` with a CUDA-event
 *                        pair recorded on the launching stream (mask 0 switches timing off).
 * sagecal_profile_read : waits for the recorded events, then fills (each host [sagecal_kernel_kinds()], may be NULL)
 *                        ms_host = summed device time per kind, timed_host = launches timed per kind (both since the
 *                        previous read), launches_host = launches per kind since load.  Returns 0 or SAGECAL_ECUDA.
 */
long long sagecal_launch_count(void);
int sagecal_kernel_kinds(void);
const char* sagecal_kernel_kind_name(int kind);
int sagecal_profile_enable(unsigned kind_mask);
int sagecal_profile_read(double* ms_host, long long* timed_host, long long* launches_host);

/*
 * The FP64 issue peak of the current device, MEASURED: a DFMA-chain kernel (8 independent chains per thread, 1024
 * threads on every SM, `iters` trips), timed with CUDA events on `stream`, best of three after a warm-up.  This is the
 * denominator of the "alu" rooflines bench.py reports ("the builder must measure a DFMA-chain peak"):
 * taken in the same run, at the clocks the compared kernels saw.  Synchronises `stream`; allocates and frees 256 B.
 * fma_per_s_host : host out, thread-level DFMAs per second (x2 = flop/s).   ms_host : host out or NULL, kernel time.
 */
int sagecal_profile_dfma_peak(int iters, double* fma_per_s_host, double* ms_host, void* stream);
/* The same for the FP64 tensor-core path: 8 independent DMMA m8n8k4 chains per warp, 16 warps per SM; FMAs per second
 * (256 per instruction).  The denominator of the station-form prediction's roofline fraction. */
int sagecal_profile_dmma_peak(int iters, double* fma_per_s_host, double* ms_host, void* stream);

/* The host-only replays of the kernels' work decompositions (test hooks) are declared in sagecal_b200_debug.h. */

#ifdef __cplusplus
}
#endif
#endif /* SAGECAL_B200_H */
