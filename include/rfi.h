/* rfi.h -- C ABI of librfi.so: the fused spectral-kurtosis + polarization-alignment
 * flag-and-average pass of arxiv 2412.14775 on one B200 (sm_100a).
 *
 * Citations are lines of /root/reference/PAPER.md ("PAPER.md:n") with the section / equation.
 *
 * The operation (one call of rfi_process_chunk), per (baseline b, channel c) "cell", per window w of
 * W = window_M consecutive time samples, per threshold set k:
 *
 *   Stokes (Eq.(2))      I = xx+yy, Q = xx-yy, U = xy+yx, V = j(xy-yx)       (all complex)
 *   SK     (Eq.(3)-(4))  S1 = sum|I_i|, S2 = sum|I_i|^2,
 *                                        tau_k = (W d_k + 1)/(W - 1) * (W S2/S1^2 - 1)
 *   DS     (Eq.(6)-(9))  for the real parts and for the imaginary parts of (Q,U,V):
 *                                        p_i = sqrt(q_i^2+u_i^2+v_i^2), r = |sum_i (q_i,u_i,v_i)/p_i| / W
 *   flag   (Eq.(5),(10))
 *                                        f_k = (tau_k < s_low_k) OR (tau_k > s_high_k) OR (r_re > gamma_k) OR (r_im > gamma_k)
 *                                        evaluated as !(tau>=s_low && tau<=s_high) || !(r_re<=gamma) || !(r_im<=gamma)
 *                                        so that a non-finite statistic flags the window
 *   excise + average  per output integration o (n_int samples): weight = number of samples in
 *                                        unflagged windows; avg = sum of those samples / weight (0 if weight = 0)
 *
 * Guards: an all-zero window has tau = -(W d + 1)/(W - 1); a sample with p_i = 0 adds the zero vector
 * (the epsilon -> 0 limit of the paper's epsilon guards).
 * Arithmetic: fp32 throughout (accumulation included); RFI_FP16 only changes the storage type of the input.
 * Eq.(5) is decided on x = tau/c against s_low/c and s_high/c (c = (W d + 1)/(W - 1) > 0; one division per threshold
 * on the host), so a decision can differ from one taken on the rounded tau only within one ulp of a threshold.
 * W = window_M, or window_M * F for T x F footprints (rfi_plan_set_window_freq).
 * rfi_plan_set_arithmetic(RFI_ARITH_TABLES) selects the paper's operation tables in per-group single/half precision instead.
 * Finite inputs must satisfy 1e-18 <= |x| <= 1e18 or x == 0 (fp32 squares must neither overflow nor
 * underflow); outside that range the statistics are unspecified (never a fault).
 *
 * Memory layouts (all device pointers unless the name starts with h_; all row-major, last index fastest):
 *   vis     [n_time][n_baselines][n_chan][4 pols: XX,XY,YX,YY][re,im]      float (RFI_FP32) or IEEE half (RFI_FP16)
 *           time-slowest "correlator dump order"; 32 B (16 B) per sample; base 16-byte aligned.
 *   avg     [K][n_out][n_baselines][n_chan][4][re,im]   float,    n_out = n_time / n_int
 *   weight  [K][n_out][n_baselines][n_chan]             uint32_t  (unflagged sample count)
 *   stats   [3][n_win][n_baselines][n_chan]             float,    planes tau (with d of set 0), r_re, r_im;
 *                                                                  n_win = n_time / window_M, w counts from chunk start
 *   flags   [K][n_win][n_baselines][ceil(n_chan/32)]    uint32_t, bit (c % 32) of word c/32, 1 = flagged;
 *                                                                  unused high bits of a baseline's last word are 0
 *
 * Ownership: the caller owns vis/avg/weight/stats and the stream; the plan owns its device threshold table,
 * its flag buffer and (for the host path) its staging buffers.  vis is never written and is read
 * once per launch: exactly once for K <= 64 threshold sets, once per 64 sets beyond that (rfi_set_thresholds).
 * rfi_process_chunk enqueues work on the stream and returns without synchronising the host.
 *
 * Errors: every function returns RFI_OK (0) or a negative code; nothing throws or aborts.
 * Threads: a plan is not internally locked; use one plan from one host thread at a time (different plans are independent).
 * Devices: a plan binds to the CUDA device that is current at its first process call (its flag buffer, class table
 * and staging buffers live there); a later process call with another device current returns RFI_EINVAL.
 */
#ifndef RFI_H_
#define RFI_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rfi_plan rfi_plan;            /* opaque host object */

enum { RFI_FP32 = 0, RFI_FP16 = 1 };         /* storage precision of vis */

enum {
    RFI_OK      =  0,
    RFI_EINVAL  = -1,   /* bad argument (shape, alignment, NULL, K < 1, d <= 0, ...) */
    RFI_ECUDA   = -2,   /* a CUDA call failed; rfi_last_cuda_error() has the text */
    RFI_ENOMEM  = -3,   /* host or device allocation failed */
    RFI_ESTATE  = -4,   /* call order: thresholds not set, no chunk processed yet, ... */
    RFI_ENODEV  = -5    /* no CUDA device / not an sm_100 device */
};

/* kernel variants (rfi_plan_set_variant); all compute the same function */
enum {
    RFI_VARIANT_AUTO   = 0,   /* the fastest measured variant for the shape (currently: direct) */
    RFI_VARIANT_DIRECT = 1,   /* per-thread 256-bit (fp32) / 128-bit (fp16) streaming loads, register double buffer */
    RFI_VARIANT_TMA    = 2,   /* warp-private TMA (cp.async.bulk.tensor) ring in shared memory */
    RFI_VARIANT_BATCHED = 3,  /* reported by rfi_plan_last_variant when K > 1 (not selectable: K decides) */
    RFI_VARIANT_TABLES = 4,   /* reported when the arithmetic mode is RFI_ARITH_TABLES */
    RFI_VARIANT_SPLIT  = 5    /* small chunks, low latency: one CTA per (tile, integration), its rows split over up to
                                 16 warps so that the whole unit is in flight at once (windows are kept small
                                 for latency).  K = 1, RFI_ARITH_FAST, time-major, n_int / block length <= 96 -- a plan in
                                 any other mode refuses the request (rfi_process_chunk: RFI_EINVAL with a message).  The SK
                                 statistic is bit-identical to the direct kernel; alignment statistics and averages are
                                 summed block-wise, i.e. equal to the other variants within the stated tolerances, not
                                 bit for bit.  Never chosen by RFI_VARIANT_AUTO. */
};

/* input layouts (rfi_plan_set_layout) */
enum {
    RFI_LAYOUT_TIME_MAJOR = 0,   /* default: vis[t][b][c][pol], correlator dump order */
    RFI_LAYOUT_CELL_MAJOR = 1    /* vis[b][c][t][pol]: each (baseline, channel) time series contiguous */
};

/* arithmetic modes (rfi_plan_set_arithmetic) */
enum {
    RFI_ARITH_FAST   = 0,     /* default: all-single reformulation (centred SK moment, exact-zero guards) */
    RFI_ARITH_TABLES = 1      /* the paper's Tables 1-2 step by step, each group in single or half precision */
};

/* One threshold set: d of Eq.(4), s_low/s_high of Eq.(5), gamma of Eq.(10)
 * (PAPER.md:103).  s_low = -inf, s_high = +inf disables the SK test; gamma = +inf disables the DS test. */
typedef struct { float d, s_low, s_high, gamma; } rfi_thresholds;

/* Create a plan for chunks of n_time samples of n_baselines x n_chan cells (N(N+1)/2 streams,
 * each mitigated separately).  Requirements (else RFI_EINVAL): n_stations >= 1; n_baselines == N(N+1)/2 or
 * N(N-1)/2; n_chan >= 1; window_M >= 2 (Eq.(4) divides by W-1); n_time % window_M == 0;
 * precision in {RFI_FP32, RFI_FP16}.  The integration length defaults to n_time (one output per chunk).
 * No window may straddle a chunk or integration boundary (no cross-chunk state).  Does not need a GPU
 * until the first process call. */
int rfi_plan_create(rfi_plan **out, int n_stations, int n_baselines, int n_chan,
                    int n_time, int window_M, int precision);

/* Samples per output integration: n_time % n_int == 0 and n_int % window_M == 0, else RFI_EINVAL. */
int rfi_plan_set_integration(rfi_plan *plan, int n_int);

/* Input layout.  RFI_LAYOUT_CELL_MAJOR reads vis[n_baselines][n_chan][n_time][4 pols][re,im] (e.g. after a corner
 * turn): the TMA kernel stages 128-byte lines (4 fp32 / 8 fp16 samples) of 32 cells through a transposing tensor
 * map, after which the arithmetic -- and therefore every output bit -- is that of the time-major TMA kernel.
 * Outputs keep their layouts; K > 1 runs the batched kernel behind the same map.  Restrictions (rfi_process_chunk
 * returns RFI_EINVAL otherwise): window_M % 4 == 0 (fp32) or % 8 == 0 (fp16), RFI_ARITH_FAST, device buffers
 * (rfi_process_chunk_host rejects it). */
int rfi_plan_set_layout(rfi_plan *plan, int layout);

/* Per-baseline threshold classes.  Every baseline stream is mitigated separately and its null
 * statistics depend on the kind of stream: an auto-correlation is Hermitian with a large constant part, so its
 * SK and alignment statistics under noise differ from a cross-correlation's (d "is given a priori").
 * n_classes = 2 assigns each baseline of the array (h_class[n_baselines], values 0/1, e.g. 0 = cross, 1 = auto;
 * copied) to a class; rfi_set_thresholds then takes K * 2 sets ordered [k][class] and every kernel decides each
 * window with the set of its baseline's class (the stats plane carries tau with the d of the cell's class).
 * n_classes = 1 (h_class ignored) restores one set per k.  Clears the thresholds: set them again afterwards.
 * RFI_EINVAL for n_classes outside {1, 2}, a NULL table or a class value above 1. */
int rfi_plan_set_baseline_classes(rfi_plan *plan, int n_classes, const uint8_t *h_class);

/* Window footprint in frequency ("a data window of size W divided into T time samples and F
 * frequency samples, W = T x F"; the paper uses 10 x 2 and 5 x 4).  T is the window_M of
 * rfi_plan_create, F defaults to 1.  With F > 1 a window covers F adjacent channels of one baseline: the
 * statistics of Eq.(3)-(4) and Eq.(6)-(9) run over all W = T*F samples (W replaces window_M in both equations),
 * the flag applies to the whole footprint, and every channel is still averaged on its own.  All
 * buffer layouts are unchanged (the F channels of a footprint carry the same statistics and flag bit).
 * RFI_EINVAL unless F is a power of two, F <= 32 and n_chan % F == 0. */
int rfi_plan_set_window_freq(rfi_plan *plan, int F);

/* Arithmetic mode.  RFI_ARITH_TABLES runs the paper's operation tables literally (Table 1, PAPER.md:131-143:
 * y = xr^2+xi^2, z = sqrt(y), s1 = sum z, s2 = sum y, tau = (Wd+1)/(W-1), s12 = s1^2, tau = tau (W s2/(s12+eps) - 1)
 * [Eq.(4) brackets], compare; Table 2: a,b,c = q^2,u^2,v^2, p = sqrt(a+b+c)+eps, q/p,u/p,v/p,
 * sums, squares, r = sqrt(q+u+v)/W, compare; once on the real and once on the imaginary parts), every operation an
 * IEEE round-to-nearest operation in the precision of its group: bit g-1 of mask14 (g = 1..7) puts Table 1 group g
 * in half precision, bit 7+g-1 Table 2 group g; eps = machine epsilon of the group's format
 * (PAPER.md:131); operands are converted into the consuming group's format.  Results are bit-identical to the
 * step-by-step CPU restatement.  Needs RFI_FP32 storage (the stream is single precision), F = 1 and
 * K = 1 (else rfi_process_chunk returns RFI_EINVAL).  Half-precision overflow yields a non-finite statistic and
 * hence a flag.  RFI_ARITH_FAST takes mask14 = 0.  RFI_EINVAL for an unknown mode or mask bits above 13. */
int rfi_plan_set_arithmetic(rfi_plan *plan, int mode, uint32_t mask14);

/* Multi-GPU sharding (every baseline stream is mitigated separately, so streams partition across
 * devices with no exchange).  Declares that this plan processes only baselines [b_first, b_first + b_count) of the
 * n_baselines given at creation: from now on every buffer (vis, avg, weight, stats, flags) holds b_count baselines
 * in place of n_baselines, in the same layouts.  RFI_EINVAL unless 0 <= b_first, b_count >= 1 and
 * b_first + b_count <= n_baselines.  Results equal the corresponding slices of an unsharded run bit for bit. */
int rfi_plan_set_baseline_shard(rfi_plan *plan, int b_first, int b_count);

/* Copy K >= 1 threshold sets from host memory (d > 0 and not NaN; s_low/s_high/gamma may be +-inf, not NaN).
 * K == 1 runs the single-set kernel; K > 1 the batched kernel that evaluates up to 64 sets in one pass over the
 * data (one launch per 64 sets; the paper tunes its thresholds with a host-side search).
 * With two baseline classes (rfi_plan_set_baseline_classes) h_sets holds K * 2 sets ordered [k][class].
 * The statistics planes (d_stats) always carry tau with the d of set 0 (of the cell's class). */
int rfi_set_thresholds(rfi_plan *plan, int K, const rfi_thresholds *h_sets);

/* On-line threshold adaptation (the thresholds follow from "the desired performance (the false alarm
 * probability)"; "some fine-tuning for each data stream is necessary ... in an online manner";
 * "dynamic adaptation of the threshold levels depending on the data streams").  The paper gives no
 * algorithm; this is a constant-false-alarm-rate rule by rank (readings A1-A6): while a chunk
 * is processed the kernel histograms tau (Eq.(4)) and max(r_re, r_im) (Eq.(9)) of every window with finite
 * statistics, per baseline class (geometric bins, 64 per octave, tau in [2^-8, 2^4), r in [2^-6, 1)); after the chunk
 * a device kernel folds them into running histograms (acc <- forget * acc + chunk) and sets the thresholds of the NEXT
 * chunk to s_low = Q_tau(beta/2), s_high = Q_tau(1 - beta/2), gamma = Q_r(1 - beta) with beta = 1 - sqrt(1 -
 * false_alarm), so that the two OR-ed detectors flag a fraction false_alarm of RFI-free data.  The first chunk runs
 * with the thresholds of rfi_set_thresholds (their d stays in force); a class with fewer than 1000 counted windows
 * keeps its thresholds.  All on the caller's stream, no host synchronisation.  false_alarm = 0 switches the
 * adaptation off.  Needs K = 1, RFI_ARITH_FAST, the time-major layout and the direct kernel (else rfi_process_chunk
 * returns RFI_EINVAL).  RFI_EINVAL unless 0 <= false_alarm < 0.5 and 0 <= forget < 1. */
int rfi_plan_set_adaptive(rfi_plan *plan, float false_alarm, float forget);

/* What the rule above costs under heavy RFI, and a bound on it (reading A8).  The histograms count every window with
 * finite statistics, contaminated ones included, so the quantiles are those of the MIXTURE: from the second chunk on
 * the detector flags about `false_alarm` of ALL windows of a stream.  While the RFI occupancy rho of the stream stays
 * below false_alarm this is conservative (a few extra flags); once rho exceeds it, the thresholds sit inside the RFI
 * distribution and at least (rho - flagged fraction) / rho of the RFI windows go unflagged.  On the paper's own
 * section-4.2 scenario (five broadband footprints, two narrowband; window-level occupancy about 0.55) the oracle
 * measures 0.73 missed detections after one update against 0.012 with the a-priori set (tests/test_adapt_oracle.py).
 * rfi_plan_set_adaptive_limit bounds the drift: an update moves a threshold at most max_loosen * |its a-priori value|
 * in the loosening direction (s_low down, s_high up, gamma up; a-priori = the set of rfi_set_thresholds or the
 * stream's row of rfi_plan_set_stream_thresholds) and any distance in the tightening direction.  max_loosen = 0 never
 * loosens; a negative value (the default) switches the bound off.  Applies from the next update on, in both scopes,
 * without restarting the adaptation.  RFI_EINVAL for NaN. */
int rfi_plan_set_adaptive_limit(rfi_plan *plan, float max_loosen);

/* Scope of the adaptation.  RFI_ADAPT_PER_CLASS (default): one pair of histograms and one threshold set per baseline
 * class, as above.  RFI_ADAPT_PER_BASELINE: "fine-tuning for each data stream" (every baseline stream is
 * mitigated separately) -- every baseline of the plan (of its shard) keeps its own running histograms and
 * its own (s_low, s_high, gamma); it starts from the a-priori set of its class and follows its own null distribution
 * from the second chunk on (same rule, readings A1-A6 with "class" read as "baseline"; a baseline contributes
 * n_chan counts per window step -- with T x F footprints every footprint is counted once per channel it covers, F
 * times, which leaves the quantiles unchanged but means the 1000-count gate is reached after 1000 / F independent
 * windows -- and keeps its thresholds while it has fewer than 1000 counts).  The streaming kernel
 * counts into a histogram private to the warp -- a 32-cell tile lies in one baseline, hence n_chan % 32 == 0 is required
 * (RFI_EINVAL from rfi_process_chunk otherwise) -- and adds it to the baseline's device histogram at the end of each
 * (tile, integration) unit; the update kernel runs one CTA per two baselines.  Restarts the adaptation. */
enum { RFI_ADAPT_PER_CLASS = 0, RFI_ADAPT_PER_BASELINE = 1 };
int rfi_plan_set_adaptive_scope(rfi_plan *plan, int scope);
/* RFI_ADAPT_PER_BASELINE only: the thresholds in force for the next chunk, h_out[n_baselines] (of the shard), and the
 * running histograms, h_out[n_baselines][768 tau bins | 384 r bins] doubles.  Both wait for the device work issued so
 * far.  RFI_ESTATE before the first chunk processed in a per-stream mode. */
int rfi_plan_get_stream_thresholds(rfi_plan *plan, rfi_thresholds *h_out);
/* Thresholds given per baseline stream by the caller (the result of an off-line fine-tuning "for each data stream",
 * PAPER.md:259): h_sets[n_baselines] (of the shard; copied; d > 0, no NaN), NULL switches the table off.  Without
 * adaptation every window of baseline b is decided with h_sets[b] (the stats plane carries tau with its d); with
 * RFI_ADAPT_PER_BASELINE the table is the a-priori state the streams start from (the per-class adaptation ignores it).
 * Same restrictions as the adaptive
 * mode (K = 1 set with rfi_set_thresholds, RFI_ARITH_FAST, time-major, direct kernel, n_chan % 32 == 0; RFI_EINVAL from
 * rfi_process_chunk otherwise, RFI_ESTATE if the shard has changed since).  rfi_plan_get_stream_thresholds returns it. */
int rfi_plan_set_stream_thresholds(rfi_plan *plan, const rfi_thresholds *h_sets);
int rfi_plan_get_stream_histograms(rfi_plan *plan, double *h_out);

/* The thresholds currently in force, one set per baseline class (h_out[n_classes], host memory): the adapted ones
 * when adaptation is on (waits for the device work enqueued so far), else set 0 of rfi_set_thresholds. */
int rfi_plan_get_thresholds(rfi_plan *plan, rfi_thresholds *h_out);

/* Diagnostics: the running histograms of the adaptation, double[2 classes][768 tau bins | 384 r bins] to host memory
 * (waits for the device work enqueued so far).  RFI_ESTATE unless adaptation is on and a chunk was processed. */
#define RFI_ADAPT_TAU_BINS 768
#define RFI_ADAPT_R_BINS 384
int rfi_plan_get_adaptive_histogram(rfi_plan *plan, double *h_out);

/* Choose a kernel variant (default RFI_VARIANT_AUTO).  RFI_EINVAL if unknown. */
int rfi_plan_set_variant(rfi_plan *plan, int variant);

/* Process one chunk resident in device memory.  d_stats may be NULL.  cuda_stream is a cudaStream_t
 * (NULL = legacy default stream).  Asynchronous.  After one warm-up call (which allocates the plan's flag buffer
 * and, for the TMA kernels, encodes the tensor map of this d_vis) a call is pure stream work -- kernel launches and
 * at most one memset -- and can be captured in a CUDA graph and replayed on the same buffers.  RFI_ESTATE if thresholds were never set; RFI_EINVAL for
 * NULL / misaligned (16 B) pointers; RFI_ECUDA if a launch failed. */
int rfi_process_chunk(rfi_plan *plan, const void *d_vis, void *d_avg, void *d_weight,
                      void *d_stats, void *cuda_stream);

/* Device pointer to the flag mask of the last processed chunk and its length in 32-bit words
 * (K * n_win * n_baselines * ceil(n_chan/32)).  Valid until the next process call or destroy; reading it is
 * ordered after the kernel only on the stream that was passed to rfi_process_chunk. */
int rfi_get_flags(rfi_plan *plan, const uint32_t **d_flags, size_t *n_words);

/* Per-set confusion counters of the last processed chunk against a ground-truth mask (BASELINE.json configs[4];
 * false-alarm / missed-detection probabilities as defined at PAPER.md:235).  d_truth: bit-packed like the flag
 * mask of ONE set, [n_win][n_baselines][ceil(n_chan/32)] uint32_t, 1 = the window of that cell carries RFI.
 * d_counts: uint64_t [K][4] = {false alarms, clean windows, missed detections, RFI windows}, counted per
 * (window, cell); zeroed and filled on the stream.  P_fa = [0]/[1], P_md = [2]/[3].  Exact integers.
 * RFI_ESTATE before the first process call; RFI_EINVAL for NULL / misaligned pointers. */
int rfi_confusion_counts(rfi_plan *plan, const uint32_t *d_truth, uint64_t *d_counts, void *cuda_stream);

/* The same counters as part of every rfi_process_chunk call (device path): with a ground-truth mask d_truth (layout as
 * above) and d_counts (uint64_t [K][4], both device pointers that must stay valid; both NULL switches it off), each
 * call zeroes d_counts on its stream and fills it for the chunk it processes.  The K-set kernel counts in the same
 * launch -- the thread that packs a (set, window) flag word compares it with the truth word, so a tuning loop
 * (false-alarm / missed-detection probabilities per candidate threshold set) needs no second pass over
 * the K masks; the other kernels are followed by the mask pass of rfi_confusion_counts on the same stream.  Same
 * exact integers either way (rfi_process_chunk_host: the mask pass after its last slab, before it returns).  Call it after rfi_set_thresholds: d_counts is sized
 * for the K of that moment, and rfi_process_chunk returns RFI_ESTATE if K has changed since.  RFI_EINVAL if exactly one
 * pointer is NULL or a pointer is misaligned (4 / 8 bytes). */
int rfi_plan_set_truth(rfi_plan *plan, const uint32_t *d_truth, uint64_t *d_counts);

/* End-to-end host path: vis in HOST memory (pinned for full speed), results to HOST memory.  Streams the
 * chunk to the device one output integration at a time on two internal streams so that host->device copies
 * overlap the kernel, then copies avg / weight / flags (and stats if non-NULL) back and synchronises.
 * Same results as rfi_process_chunk. */
int rfi_process_chunk_host(rfi_plan *plan, const void *h_vis, void *h_avg, void *h_weight,
                           void *h_flags, void *h_stats);

int rfi_plan_destroy(rfi_plan *plan);

/* ---------------------------------------------------------------------------------------------------------------
 * The reinforcement-learning environment of section 3: one launch evaluates
 * n_windows windows against ONE 14-bit precision mask (bit g-1: Table 1 group g in half; bit 7+g-1: Table 2 group g)
 * so that an external soft-actor-critic loop (host side, out of scope) gets state, cost and reward for its batch.
 *   d_windows  [n_windows][W][4 pols][re,im] float: each window's W = T x F samples contiguous (the
 *              tables do not use the order of the samples beyond the order of their sums)
 *   d_out      [n_windows][RFI_RL_RECORD_DOUBLES] double:
 *              [0..9]   data features: log(sum_i part(X_i)^p)/W for (I,2), (I,4), (Q,2), (U,2), (V,2), real parts then
 *                       imaginary parts, natural log, on the single-precision Stokes parameters
 *              [10..23] the 14 precision bits
 *              [24..44] the 21 errors: per group, mean over the group's outputs of |value in the chosen precisions -
 *                       value with every operation in double| (+inf if not finite): Table 1 groups 1-7, Table 2 on the
 *                       real parts groups 1-7, Table 2 on the imaginary parts groups 1-7 (group 7 of Table 2: the flag)
 *              [45]     operation cost: cost column x C, C = 1 single / 0.6 half: Table 1 as printed
 *                       (3W, W, W, W, 1, 1, 1+2), Table 2 groups 1-7 = 3W, W, 3W, 3W, 3, 4, 1, counted twice
 *              [46]     type conversions (0.3 each): elements carried over data-flow edges whose ends differ in format
 *              [47],[48] overflow / underflow events (exact result finite but rounded not; exact non-zero but rounded
 *                       below the smallest normal number of the format)
 *              [49]     how many of the three flags (SK, DS real, DS imaginary) equal the double-precision flags
 *              [50]     reward = reward_per_match * [49] - [45] - 0.3 * [46] - 20 * ([47] + [48] > 0)     (
 *                       the printed reward constant is garbled, hence the argument)
 *              [51]     flags: mixed-precision (bit 0 SK, 1 DS real, 2 DS imaginary) + 8 * double-precision flags
 * Thresholds (d, s_low, s_high, gamma) are read from host memory.  Every operation is an IEEE round-to-nearest
 * operation of its group's format; eps = machine epsilon of the format (2^-52 for the ground truth); results equal the
 * step-by-step CPU restatement (bit for bit except the libm-dependent logarithms of the features).  Asynchronous on the
 * stream.  RFI_EINVAL for NULL / misaligned pointers, W < 2, mask bits above 13, d <= 0. */
#define RFI_RL_RECORD_DOUBLES 52
int rfi_rl_evaluate(const float *d_windows, int64_t n_windows, int W, uint32_t mask14,
                    const rfi_thresholds *h_thr, double reward_per_match, double *d_out, void *cuda_stream);
/* The same with one precision mask PER WINDOW: d_masks[n_windows] uint16_t on the device (bits 0-13; higher bits are
 * ignored) -- a batch of (state, action) pairs, as a vectorised environment or a replay batch of the agent produces
 * them (the action selects the precision of every group).  Record n equals what rfi_rl_evaluate
 * gives for window n with mask d_masks[n].  RFI_EINVAL for a NULL / misaligned d_masks. */
int rfi_rl_evaluate_masks(const float *d_windows, int64_t n_windows, int W, const uint16_t *d_masks,
                          const rfi_thresholds *h_thr, double reward_per_match, double *d_out, void *cuda_stream);

/* ---------------------------------------------------------------------------------------------------------------
 * Section-4.2 simulator: seeded synthetic blocks with injected RFI at a set
 * interference-to-noise ratio, generated on the device.  One realisation = one simulated baseline = n_time x n_chan
 * time-frequency samples (the paper: 2000 x 512, "about 1 s of data with about 200 kHz bandwidth");
 * realisations sit on the baseline axis: d_vis is vis[n_time][n_real][n_chan][4][re,im] float, i.e. a chunk for a
 * plan with n_baselines = n_real.  Per realisation (readings S1-S9 in DESIGN.md section 2):
 *   noise     a * e_p e_q^H + sky: e_p, e_q ~ CN(0, I_2) station voltages per sample ("the conjugate product of the
 *             two voltages"), sky ~ CN(0,1) per correlation, a = 100 U(0,1) constant over the block
 *   sources   n_sources (200): (u,v,w) = 300 N(0,1); (l,m) ~ U(-0.5,0.5), n = sqrt(1-l^2-m^2); flux ~ U(1,10);
 *             coherence flux * exp(j 2 pi f (ul+vm+w(n-1))/c), f_k = 120 MHz + k * 200 kHz / n_chan; unpolarised
 *             (xx = yy = half the coherence, Eq.(2) has no 1/2), constant in time
 *   RFI       n_broadband footprints [t0,t1) x [c0,c1) (sorted uniform edges) filled with ones; n_narrowband: one
 *             channel, all times, exp(j 2 pi t / P), P = max(120 U(0,1), 2) samples; n_narrowdur: one time sample,
 *             all channels, exp(j 2 pi c / P), P = max(1024 U(0,1), 2); each scaled by J/||J||, J = 4 draws of
 *             CN(0,1) = (xx,xy,yx,yy); draws whose coherency J J^H (J as a 2x2 matrix) is more than 90 % polarised
 *             are redrawn (<= 16 times); polarized = 0: J = (1,0,0,1)/sqrt(2) (Fig. 3(b))
 *   mixing    data = celestial + g * rfi, g^2 = inr * P_celestial / P_rfi, P = total power over the block and the
 *             four correlations; inr = 0 adds nothing
 * d_truth (nullable): the window-level ground truth for rfi_confusion_counts, bit-packed like one
 * set of the flag mask, [n_time/window_T][n_real][ceil(n_chan/32)]: bit c is set where the window_T x window_F
 * footprint containing channel c holds an RFI point (needs window_T | n_time, window_F | n_chan).
 * d_table / d_sources (nullable, diagnostics and tests): the per-realisation parameter table and the source coherence
 * double[n_real][n_chan][re,im]; when NULL, work buffers are allocated internally and the call synchronises the stream,
 * otherwise it only enqueues work.  Random numbers: Philox-4x32-10 keyed by `seed`, counter (index, 0, stream,
 * realisation) -- every value is a pure function of its coordinates (the draw table is in oracle/sim42_oracle.py and
 * csrc/rfi_sim42.cu).  The Gaussian transform of the noise runs in fp32, parameters and RFI phases in fp64.
 * RFI_EINVAL (with rfi_last_cuda_error text) for sizes < 1, n_real > 65535, n_sources > 4096, more than
 * RFI_SIM42_MAX_COMPONENTS RFI components, a negative or non-finite inr, a misaligned d_vis. */
#define RFI_SIM42_MAX_COMPONENTS 16
typedef struct {
    int n_time, n_chan, n_real;                    /* block size and number of realisations */
    int n_sources;                                 /* 200 in the paper */
    int n_broadband, n_narrowband, n_narrowdur;    /* 5, 1, 1: "five broadband ... and two narrowband" (Fig. 2) */
    int polarized;                                 /* 1: random J with the 90 % cut; 0: unpolarised RFI */
    float inr;                                     /* interference-to-noise ratio (total power ratio) */
    int window_T, window_F;                        /* footprint of the truth mask */
    uint64_t seed;
} rfi_sim42_config;
typedef struct {
    int kind;                                      /* 0 broadband, 1 narrowband (one channel), 2 narrow duration (one sample) */
    int t0, t1, c0, c1;                            /* support [t0,t1) x [c0,c1) */
    int tries;                                     /* J draws used (0 when unpolarised) */
    double period;                                 /* samples; 0 for broadband */
    double J[8];                                   /* J / ||J||: xx, xy, yx, yy as (re, im) */
} rfi_sim42_component;
typedef struct {
    double a, u, v, w;                             /* receiver-noise scale; baseline coordinates (m) */
    double p_cel, p_rfi, gain;                     /* total powers and g of the mixing step */
    int n_comp, reserved;
    rfi_sim42_component comp[RFI_SIM42_MAX_COMPONENTS];
} rfi_sim42_realisation;
int rfi_sim42_generate(const rfi_sim42_config *cfg, void *d_vis, uint32_t *d_truth,
                       rfi_sim42_realisation *d_table, double *d_sources, void *cuda_stream);
size_t rfi_sim42_vis_bytes(const rfi_sim42_config *cfg);      /* n_time * n_real * n_chan * 32 */
size_t rfi_sim42_truth_bytes(const rfi_sim42_config *cfg);    /* (n_time/window_T) * n_real * ceil(n_chan/32) * 4 */

/* rfi_sim42_generate for callers that cannot allocate device memory.  The generator needs two work arrays between its
 * kernels (parameter table, source coherence).  rfi_sim42_generate either allocates them on every call (cudaMalloc +
 * cudaFree, both of which serialise with all streams of the device) or takes them from the caller.  Neither suits code
 * that lives inside another program's memory budget: a plug-in of a correlator / beam-former process that partitioned
 * the whole GPU at start-up and passes only each call's input and output buffers, or a tuning loop generating fresh
 * section-4.2 blocks beside live flagging streams that an allocation would stall.  This entry point keeps the work
 * arrays in a fixed array inside the library image instead and calls no cudaMalloc, cudaFree or other allocating
 * routine -- the caller passes only the configuration and the outputs:
 *   d_vis, d_truth (nullable), cuda_stream: as for rfi_sim42_generate; same kernels, same draws, so the same output
 *   (bit for bit where inr = 0; otherwise equal up to the summation order of the two power totals, which are
 *   accumulated with floating-point atomics in either entry point).  Only enqueues work; does not synchronise.
 * Limits: n_real <= RFI_SIM42_STATIC_MAX_REAL and n_real * n_chan <= RFI_SIM42_STATIC_MAX_CELLS (the paper's 400-run
 *   sweep at 512 channels fits); larger requests are refused with RFI_EINVAL and a message in
 *   rfi_last_cuda_error -- split the batch over calls (realisation r of a call with seed s depends on (s, r) only).
 * Cost: the array (rfi_sim42_static_bytes(), about 4.8 MiB) occupies every GPU that loads the library until the
 *   process exits, used or not.
 * First call on a device: looks up the array's address on that device (the current device; one cudaGetSymbolAddress,
 *   which may make the runtime load the module there).  Make that first call before any stream capture begins.
 * Sharing: all calls on a device use the same array and find the previous call's contents in it.  Nothing needs
 *   clearing by the caller -- the first kernel rewrites every table row it uses, accumulators included -- but two
 *   calls that can overlap on the GPU (different streams without an ordering between them, or two host threads)
 *   race on it and corrupt each other: order them, e.g. issue them on one stream.
 * d_vis must be memory of the current device (RFI_EINVAL otherwise); the stream must belong to it too. */
#define RFI_SIM42_STATIC_MAX_REAL 512
#define RFI_SIM42_STATIC_MAX_CELLS 262144
int rfi_sim42_generate_static(const rfi_sim42_config *cfg, void *d_vis, uint32_t *d_truth, void *cuda_stream);
size_t rfi_sim42_static_bytes(void);                           /* size of the built-in work array, per GPU */

/* Diagnostics (not part of the method): read-only streaming bandwidth of the current device.  Reads `bytes` (>= 32,
 * a multiple of 32 is used) of the 32-byte aligned device buffer d_buf once per launch with the 256-bit streaming
 * load of the direct kernel, `repeats` timed launches after two warm-up launches, CUDA events on the stream;
 * *h_ms_best (host) receives the best launch time in milliseconds.  Synchronises the stream.  The flag-and-average
 * pass is a one-touch read stream (the correlator output is read once and averaged down), so this is
 * the like-for-like denominator for its achieved GB/s; MEASURED_PEAKS.json's figure is a read+write copy. */
int rfi_probe_read_bandwidth(const void *d_buf, size_t bytes, int repeats, float *h_ms_best, void *cuda_stream);

/* Diagnostics (not part of the method): the same for the traffic MIX of a K-set pass (batched-threshold mode, K sets of
 * averaged outputs per chunk: 32 B in and K * (36/n_int + 1/(8 W)) B out per sample): every warp reads
 * `reads_per_write` 1 KiB rows of d_in with the streaming load and then writes one 1 KiB row of d_out with an
 * evict-first 256-bit store, no arithmetic.  d_in, d_out: 32-byte aligned device buffers; floor(in_bytes /
 * (reads_per_write KiB)) KiB of d_out are written (RFI_EINVAL if out_bytes is smaller, or nothing would be read);
 * *h_ms_best (host): best of `repeats` timed launches over four launch shapes, *h_bytes_moved (host, may be NULL):
 * bytes read + written per launch.  Synchronises the stream.  What this reaches is the ceiling for the batched
 * kernels: HBM serves a 90/10 read/write mix more slowly than a pure read stream. */
int rfi_probe_mix_bandwidth(const void *d_in, size_t in_bytes, void *d_out, size_t out_bytes, int reads_per_write,
                            int repeats, float *h_ms_best, size_t *h_bytes_moved, void *cuda_stream);

/* helpers */
const char *rfi_strerror(int code);
const char *rfi_last_cuda_error(void);                 /* detail text of the last failed process call of this thread: the
                                                          CUDA error string, or which shape rule an RFI_EINVAL broke;
                                                          cleared at the start of every rfi_process_chunk* call */
size_t rfi_flags_bytes(const rfi_plan *plan);          /* bytes of the flag mask for the current K */
size_t rfi_avg_bytes(const rfi_plan *plan);            /* bytes the caller must provide for d_avg */
size_t rfi_weight_bytes(const rfi_plan *plan);
size_t rfi_stats_bytes(const rfi_plan *plan);
size_t rfi_vis_bytes(const rfi_plan *plan);
uint64_t rfi_plan_launch_count(const rfi_plan *plan);  /* kernels launched by this plan so far */
int rfi_plan_last_variant(const rfi_plan *plan);       /* variant the last process call used */
const char *rfi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RFI_H_ */
