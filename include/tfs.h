/* tfs.h -- C ABI of libtfs: batch evaluation of the semi-coherent time-frequency detection
 * statistic Upsilon_Nseg on one NVIDIA B200 (sm_100a).
 *
 * Method: arXiv 2510.19047, "Global time-frequency search for stellar-mass binary black holes
 * in LISA".  Citations "P:<n>" are line numbers of the paper text with the equation
 * they fall in; "C<n>" are the readings listed in DESIGN.md section 3.
 *
 * What one call of tfs_eval computes, for every template theta_i of a batch:
 *   track   f_m, fdot_m, phi_m, A_m at each tranche start t_m = m*DT        (Eqs. 12-15)
 *   pixels  h~_m(f_k)/DT in the window k_lo..k_hi around f_m, Fresnel kernel (Eqs. 16-22)
 *   sums    z_n  = sum_alpha T_alpha sum_{m in seg n} sum_k g[m] W conj(D) h~  (Eq. 31, Eq. 30)
 *           hh_n = sum_alpha |T_alpha|^2 sum_m sum_k g[m] W |h~|^2
 *   result  P_n = |z_n|^2 / hh_n (0 if hh_n = 0),  Upsilon = sum_n P_n         (Eq. 8, Eq. 9)
 * with n(m) = floor(m*N_seg/Nt) (C9) and W = 4 df / S in the data's units so that noise has
 * E|D|^2 = 2/W (absorbs the 4 and delta-f of Eqs. 1 and 7).
 *
 * Geometry (C1): Nt tranches of length DT = 2*Nf*dt; Nf frequency bins of width df = 1/DT;
 * bin k sits at f_k = k*df.  All arrays are C-contiguous, frequency fastest.
 *
 * Every step runs in CUDA kernels of this library; there is no CPU fallback.  All functions
 * return 0 on success or a negative TFS_E* code; nothing throws or aborts across the ABI.
 * Pointers marked "host or device" are classified with cudaPointerGetAttributes; the caller
 * owns every array it passes and the library never keeps a caller pointer after the call
 * returns (device-pointer work is only ENQUEUED on `stream`: the caller must keep those
 * arrays alive and unchanged until it has synchronised that stream).  Host outputs imply a
 * stream synchronisation inside the call.  A context must not be used from two threads at once, and
 * its calls share scratch buffers: work enqueued on one stream must have completed (or be ordered
 * before) the next call on another stream; tfs_upload_data / tfs_upload_timeseries must not be
 * called while a tfs_eval of the same context is still running.
 * CUDA graphs: after one warm-up call with the same shapes and N_seg (scratch buffers and the piece table then exist),
 * tfs_eval / tfs_eval_tf / tfs_eval_tseg / tfs_topk / tfs_refine* with DEVICE buffers only enqueue kernels and memsets --
 * no allocation, copy or synchronisation -- and can be captured into a CUDA graph (stream capture) and replayed.
 * A captured graph holds raw device addresses of context-owned memory (scratch buffers, the cached piece table of its
 * (N_seg, seg_tranches), the data grid and its TMA descriptors).  They stay valid only while the context is left as the
 * capture found it.  RE-CAPTURE the graph (after a new warm-up call) whenever one of these happened since:
 *   - any tfs_upload_data / tfs_upload_timeseries on the context (the grid is rewritten, every piece table is dropped);
 *   - any call on the context with a larger n, larger N_seg * n, more knots or other outputs than the captured one
 *     (a scratch buffer may have been freed and re-allocated larger);
 *   - calls with more than 64 distinct (N_seg, seg_tranches) pairs since the last upload (the piece-table cache is then
 *     emptied and rebuilt);
 *   - tfs_destroy.
 * Replaying a stale graph reads freed or re-laid-out memory; the library cannot detect it.
 */
#ifndef TFS_H
#define TFS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define TFS_API __attribute__((visibility("default")))
#else
#define TFS_API
#endif

#define TFS_OK       0
#define TFS_EINVAL  -1   /* bad shape / N_seg<1 / N_seg>Nt / k<1 / k>n / NULL required pointer / unsupported option */
#define TFS_ESTATE  -2   /* tfs_eval or tfs_count_pixels before tfs_upload_data */
#define TFS_ENOMEM  -3   /* host or device allocation failed */
#define TFS_ECUDA   -4   /* CUDA runtime error; text in tfs_last_error */

#define TFS_PARAM_COLS 8 /* doubles per template row, see tfs_eval */

typedef struct tfs_ctx tfs_ctx;   /* opaque; owns every device buffer it allocates */

/* Options; pass NULL to tfs_create for the defaults.  A zero-initialised struct is NOT the
 * default set: fill it with tfs_default_opts first. */
typedef struct {
  int    half_width;     /* H: window reaches H bins below ceil(f_m/df); default 10 -> N_F = 21 (C3)   */
  int    adaptive_width; /* 1 (default): k_hi = ceil((f_m + fdot_m DT)/df) + H (C4); 0: paper-strict ceil(f_m/df)+H */
  double c_max;          /* tranches with fdot_m*DT^2 > c_max are skipped; default 300 (C4)              */
  double f_lo, f_hi;     /* band [Hz]: tranche active iff f_lo <= f_m and f_m + fdot_m DT <= f_hi;
                            <= 0 means the default [1*df, (Nf-1)*df]                                           */
  int    fresnel_mode;   /* 0 (default): Fresnel auxiliary functions accurate to ~1e-7;
                            1: the paper's approximants Eqs. 23-28 verbatim (C8)                    */
  int    weight_mode;    /* 0 (default): tfs_upload_data looks for separable weights W[a,m,k] = a[m] b[k]
                            (PSD per tranche x PSD shape; C11) and then reads no per-pixel
                            weight in the hot loop; 1: always treat W as a general per-pixel array            */
  int    basis;          /* 0 (default): the paper's grid, complex short-time Fourier tranches with the
                            Fresnel-kernel template (Eq. 16).  1: real-coefficient orthonormal WDM wavelet pixels
                            (BASELINE.json north_star's wording; the paper only cites wavelet methods):
                            Nt time pixels of duration Nf*dt x Nf layers of width 1/(2 Nf dt), `coeff` is then
                            [C][Nt][Nf] REAL floats, C <= 2, the track is expanded about the pixel centre and the
                            template pixel is the Meyer window's chirp response (readings W1-W7);
                            per segment the statistic is maximised over amplitude and phase with the 2x2 Gram matrix
                            of the two template quadratures; seg_dh = (a, b), seg_hh = (hcc + hss)/2                  */
  int    wdm_half_width; /* basis 1: layers kept on either side of the two the track sits between; default 2 (W5)    */
  double wdm_kappa_max;  /* basis 1: pixels with 4 fdot (Nf dt)^2 above this are skipped; default 8 (W7)              */
  double tukey_alpha;    /* 0 (default): the template pixel is Eq. 16 as printed, the transform of the un-windowed
                            tranche.  alpha in [1e-3, 1]: window-aware template for data whose tranches were multiplied by a
                            Tukey window of shape parameter alpha before their FFT ("Tukey-windowed with a shape
                            parameter of 0.1"; tfs_upload_timeseries): Eq. 16's integrand times the continuous window
                            w(s), s = t/DT in [0, 1] (cosine tapers of length alpha/2 at both ends; readings C2, C24):
                                h~_w(f_k)/DT = A e^{i phi} int_0^1 w(s) exp{i (2 pi u s + pi c s^2)} ds,  u = x - k,
                            evaluated in closed form (Fresnel auxiliary functions at the taper ends and at u +- 1/alpha).
                            Window, activity and segment rules are unchanged.  Basis 0 and fresnel_mode 0 only; every
                            item then takes the global-memory gather kernel (about 10x the cost of the default)            */
} tfs_opts;

TFS_API void tfs_default_opts(tfs_opts* opts);

/* Create a context for an Nt x Nf grid sampled at dt seconds with n_channels TDI channels
 * (Eq. 3 sums alpha = 1..3; the paper uses A, E, T; BASELINE.json's configs use A, E):
 * n_channels = 1, 2 or 3.  Channels are stored in pairs (0, 1) and (2, -); an odd last channel costs
 * as much as a pair.  Uses the current CUDA device, which must also be current in every later call on
 * this context (TFS_ESTATE otherwise).  Nt <= 2000000 and Nt*(Nf+16) < 2^31.
 * *out is set to NULL on failure (the reason is then in tfs_last_error(NULL)). */
TFS_API int tfs_create(tfs_ctx** out, int Nt, int Nf, double dt, int n_channels, const tfs_opts* opts);

/* Upload (copy + repack) the TF data product.
 *   coeff    [C][Nt][Nf][2] float, (re, im) of D[alpha, m, k]          host or device, required
 *   weight   [C][Nt][Nf]    float, W >= 0 per pixel (C11)               host or device, NULL => 1
 *   gap_mask [Nt]           uint8, 1 = valid, 0 = tranche overlaps a gap (C10); NULL => all valid
 * The library keeps its own repacked copy (Y = W*D interleaved by channel, and W, both transposed
 * to time-contiguous [k][m]) plus the compacted list of valid tranches, and classifies the weights
 * (tfs_weight_structure).  A pixel whose W*D or W is not finite gets weight 0.  May be called again
 * to replace the data.  Synchronises `stream` before returning. */
TFS_API int tfs_upload_data(tfs_ctx* ctx, const float* coeff, const float* weight,
                    const uint8_t* gap_mask, void* stream);

/* Time-series front end (the step before the path): window every tranche of N = 2*Nf samples
 * with a Tukey window of shape parameter tukey_alpha (the paper uses 0.1; 0 = boxcar), Fourier-transform
 * it, attach the noise weights of a one-sided PSD model and turn sample gaps into the tranche mask; then
 * proceed exactly as tfs_upload_data:
 *     D[a,m,k] = (1/N) sum_n w[n] x[a, m*N + n] exp(-2 pi i k n / N),   k = 0 ... Nf-1
 *                (= dt*DFT/DT: the continuous-FT convention with the common factor DT dropped, C16)
 *     W[a,m,k] = 4*DT / S_a[k]   (0 where S is not positive and finite; 1 everywhere if psd == NULL),
 *                so that E[W |D|^2] = 2 <w^2> for noise of that PSD
 *     g[m]     = 1 iff every sample of tranche m is valid (sample_mask) and finite (a NaN/Inf sample drops its tranche, C20)
 *   x           [C][Nt*2*Nf] float, real TDI series at cadence dt            host or device, required
 *   sample_mask [Nt*2*Nf]    uint8, 1 = valid sample; NULL => all valid        host or device
 *   psd         [C][Nf]      float, one-sided PSD [1/Hz] at f_k = k/DT; NULL => W = 1   host or device
 *   coeff_out [C][Nt][Nf][2], weight_out [C][Nt][Nf], gap_out [Nt]: nullable copies of D, W, g
 *                (host or device), e.g. to draw the whitened spectrogram of Fig. 3
 * These weights are separable by construction (one PSD model per channel), so with weight_mode = 0 the library takes
 * the per-bin table b_a[k] = 4 DT / S_a[k] directly (tfs_weight_structure 1, or 2 without a PSD): the per-pixel array
 * W is only materialised when weight_out is given, weight_mode = 1 or fresnel_mode = 1 (whose kernel reads per-pixel weights).
 * Nf must factor into 2, 3 and 5 (shared-memory FFT) and be <= 12800; basis 0 only.  Synchronises `stream`. */
TFS_API int tfs_upload_timeseries(tfs_ctx* ctx, const float* x, const uint8_t* sample_mask, const float* psd,
                                  double tukey_alpha, float* coeff_out, float* weight_out, uint8_t* gap_out,
                                  void* stream);

/* Evaluate Upsilon_{N_seg} for n templates.
 *   params  [n][8] double: Mc [Msun], tc [s after data start], phic [rad],
 *                          T_A.re, T_A.im, T_E.re, T_E.im (Eq. 29, constant per template, C5),
 *                          amp (A_m = amp * f_m^(2/3))                   host or device, required
 *   template model: 0PN chirp (C5): M = Mc*GMsun/c^3, tau = tc - t_m (> DT), X = tau/(5M),
 *     f = X^(-3/8)/(8 pi M), phi = phic - 2 X^(5/8), fdot = 3 f/(8 tau).
 *   upsilon   [n]           float   required      host or device
 *   seg_power [n][N_seg]    float   nullable      P_n
 *   seg_dh    [n][N_seg][2] float   nullable      (re, im) of z_n
 *   seg_hh    [n][N_seg]    float   nullable      hh_n
 * 1 <= N_seg <= Nt.  Rows containing NaN/Inf or Mc <= 0 yield zeros and are counted
 * (tfs_bad_param_count), not fatal.  n == 0 is a no-op.  Arithmetic: fp64 track, fp32 pixels,
 * fp32 sums within a piece (<= 64 tranches of one segment), fp64 across pieces and segments, fp32 stores.
 * On a 1-channel context T_E is ignored.  The row has no column for a third channel: on a 3-channel context tfs_eval
 * (and tfs_eval_tseg) return TFS_EINVAL until the caller has stated T_T with tfs_set_third_channel_factor, so that the
 * paper's A, E, T sum (Eq. 3) never silently becomes a two-channel statistic. */
TFS_API int tfs_eval(tfs_ctx* ctx, const double* params, long long n, int N_seg,
             float* upsilon, float* seg_power, float* seg_dh, float* seg_hh, void* stream);

/* The third channel's transfer factor for tfs_eval / tfs_eval_tseg on a 3-channel context: one complex constant T_T for
 * every template of the following calls (kept until set again).  (0, 0) is allowed and means "leave channel T out on
 * purpose": the evaluation then costs what a 2-channel context costs; any other value adds a pass over the third
 * channel.  Per-template or frequency-dependent factors go through tfs_eval_tf, which ignores this constant.
 * TFS_EINVAL on a context with fewer than 3 channels or for a non-finite value. */
TFS_API int tfs_set_third_channel_factor(tfs_ctx* ctx, double re, double im);

/* The same evaluation with a frequency-dependent transfer factor per template (Eq. 7 and P:213 Eq. 29:
 * T_alpha(f_nm), "computed once per tranche for all frequency bins"): template i carries, for each of the
 * context's C channels, a table of n_knots complex values at the frequencies f_knot0 + j*f_knot_step; the factor
 * of tranche m is the table interpolated linearly at f_m (the tranche-start frequency, C6), held at the end
 * values outside the knots; n_knots == 1 means one constant per channel.  The columns T_A, T_E of `params` are
 * then ignored (they must still be finite).  This is also how the third channel gets a per-template transfer factor:
 * tfs_eval on a 3-channel context uses T_A, T_E of `params` and the one constant of tfs_set_third_channel_factor.
 *   transfer [n][C][n_knots][2] float (re, im)       host or device, required
 *   1 <= n_knots <= 65536; f_knot_step > 0 [Hz] when n_knots > 1.
 * The factors are applied in fp32 once per tranche; everything else is as in tfs_eval. */
TFS_API int tfs_eval_tf(tfs_ctx* ctx, const double* params, long long n, int N_seg,
                const float* transfer, int n_knots, double f_knot0, double f_knot_step,
                float* upsilon, float* seg_power, float* seg_dh, float* seg_hh, void* stream);

/* The same evaluation with segments of FIXED DURATION T_seg = seg_tranches * DT laid from the start of the data,
 * t_n = n T_seg ("the n-th segment covers [t_n, t_n+1], t_n = n T_seg"; P:57 M_tr = T_seg/DT tranches per segment):
 * n(m) = floor(m / seg_tranches), N_seg = ceil(Nt / seg_tranches) segments, the last one shorter when seg_tranches does
 * not divide Nt (tfs_eval's equal-index rule, reading C9, is the same thing whenever N_seg divides Nt).
 *   n_seg_eff [n] int32, nullable: the number of segments in which template i has signal (hh_n > 0).  This is the
 *             paper's template-dependent "total number of segments" N_seg = tau / T_seg, tau = min(T_obs, t_c),
 *             counted on the grid: segments past the merger, outside the band or wholly inside gaps do not count.  For
 *             pure noise E[Upsilon] = 2 n_seg_eff, so it is what a threshold on Upsilon has to be scaled with.
 *   seg_power [n][N_seg], seg_dh [n][N_seg][2], seg_hh [n][N_seg] with N_seg = ceil(Nt / seg_tranches); nullable.
 * 1 <= seg_tranches (values >= Nt give one segment).  Everything else as tfs_eval. */
TFS_API int tfs_eval_tseg(tfs_ctx* ctx, const double* params, long long n, int seg_tranches,
                          float* upsilon, int* n_seg_eff, float* seg_power, float* seg_dh, float* seg_hh, void* stream);

/* Top-k of a batch (BASELINE.json north_star (3); the optimiser keeps the best parameter sets of each
 * iteration).  Indices and values of the k largest entries of upsilon[0..n), descending; equal values are
 * ordered by lower index first; NaN sorts below everything.  1 <= k <= n.
 *   upsilon host or device;  idx [k] int64 and val [k] float, host or device, required. */
TFS_API int tfs_topk(tfs_ctx* ctx, const float* upsilon, long long n, int k,
             long long* idx, float* val, void* stream);

/* tfs_topk for callers that must not allocate device memory.
 *
 * Who this is for: code that runs where cudaMalloc / cudaFree are off limits -- a plug-in handed a fixed memory
 * budget by its host application (an inference server or pipeline stage that owns the whole device heap and forbids
 * growth after start-up), a latency-critical loop that cannot tolerate the implicit device synchronisation of
 * cudaMalloc/cudaFree, or a process whose memory pool is already full.  Every other call of this library needs a
 * tfs_ctx, and tfs_create, tfs_upload_* and the first call of each size allocate; this one needs no context and
 * never calls cudaMalloc, cudaFree or any allocating library routine.
 *
 * What it computes: exactly what tfs_topk computes (same kernels, same order: descending value, equal values by
 * lower index, NaN last), so idx/val are bit-identical to tfs_topk's.
 *   upsilon [n] float, idx [k] int64, val [k] float: DEVICE pointers only (a host pointer would need a staging
 *   buffer, i.e. an allocation) -> TFS_EINVAL otherwise.  The caller owns all three.
 *   1 <= n < 2^32;  1 <= k <= min(n, TFS_TOPK_STATIC_MAX_K).  A larger k is rejected with TFS_EINVAL and a message
 *   naming the limit (tfs_last_error(NULL)); use tfs_topk for those.
 * Work is only enqueued on `stream`; nothing is synchronised.
 *
 * Where the scratch lives: the radix-select state (1 KiB) and the 2^ceil(log2 k) sort keys (8 B each) sit in one
 * array of fixed size compiled into the library (TFS_TOPK_STATIC_MAX_K * 8 + 2048 bytes = 514 KiB).  Every GPU on
 * which a process loads libtfs.so holds that array from load until exit, used or not.
 *
 * First call on each device: it looks up the array's device address (once per device, with that device current)
 * and the SM count, and caches them.  Make that first call outside any stream capture.
 *
 * Sharing: there is ONE array per device, shared by every caller and every stream in the process, and it keeps
 * whatever the previous call left.  Each call re-initialises the parts that must start from zero (histogram,
 * counters, padding keys) on `stream` before using them, so calls issued one after another on the same stream are
 * independent.  Two calls whose kernels can overlap on the GPU (different streams without an event between them,
 * or two host threads) race on the array and return garbage: order them yourself. */
#define TFS_TOPK_STATIC_MAX_K 65536
TFS_API int tfs_topk_static(const float* upsilon, long long n, int k, long long* idx, float* val, void* stream);

/* Ladder refinement (BASELINE.json configs[4]; the hierarchical N_seg reduction of P:104, P:347;
 * reading C19 of DESIGN.md).  For each of the k survivors j (row idx[j] of params) write r*r
 * children on a lattice r times denser per dimension that tiles the parent's (Mc, tc) cell of
 * size (Mc*d_mc_rel) x d_tc:
 *     o_i = (2 i + 1 - r) / (2 r),  i = 0..r-1            (r = 4: -3/8, -1/8, 1/8, 3/8)
 *     child (a, b):  Mc' = Mc * (1 + o_a * d_mc_rel),  tc' = tc + o_b * d_tc,  other columns copied,
 * stored at row j*r*r + a*r + b of children.  fp64, every product and sum rounded separately, so
 * the result is bit-reproducible.  An idx[j] outside [0, n) yields a row of NaN (which tfs_eval
 * scores 0 and counts as bad).
 *   params   [n][8] double, host or device;  idx [k] int64, host or device (tfs_topk's output)
 *   children [k*r*r][8] double, host or device, required;  1 <= r <= 64;  k == 0 is a no-op. */
TFS_API int tfs_refine(tfs_ctx* ctx, const double* params, long long n, const long long* idx, long long k,
               int r, double d_mc_rel, double d_tc, double* children, void* stream);

/* Tile search (the paper tiles the search volume in (Mc, f_in), f_in = f(t_0 = 0): tiles of 5 Msun x
 * 1e-4 Hz below and 1e-3 Hz above 10 mHz, and maximises the statistic in each tile).
 * tfs_tile_lattice writes the cell-centred n_mc x n_fin lattice of the tile [mc_lo, mc_hi] x [fin_lo, fin_hi]:
 *     row i*n_fin + j:  Mc = mc_lo + (i + 1/2) d_mc,  f_in = fin_lo + (j + 1/2) d_fin,
 *                       tc = tau(Mc, f_in) = 5 M (8 pi M f_in)^(-8/3),  M = Mc G Msun/c^3   (t_c = remaining lifetime, P:57;
 *                       the inverse of tfs_eval's 0PN track at t = 0), columns 2..7 copied from row[2..7],
 *     d_mc = (mc_hi - mc_lo)/n_mc,  d_fin = (fin_hi - fin_lo)/n_fin.
 *   row [8] double, HOST pointer;  params [n_mc*n_fin][8] double, host or device.  n_mc*n_fin < 2^31.
 * tfs_refine_fin is tfs_refine carried out in (Mc, f_in): survivor j (row idx[j] of params) is replaced by r*r
 * children that tile its (d_mc x d_fin) cell,
 *     f_in = f(tc) = (tc/5M)^(-3/8)/(8 pi M);  child (a, b):  Mc' = Mc + o_a d_mc,  f_in' = f_in + o_b d_fin,
 *     tc' = tau(Mc', f_in'),  o_i = (2 i + 1 - r)/(2 r),  other columns copied;  row j*r*r + a*r + b of children.
 * Lattice positions use separately rounded fp64 products and sums; tau and f go through pow (a few ulp).
 * Arguments otherwise as tfs_refine. */
TFS_API int tfs_tile_lattice(tfs_ctx* ctx, double mc_lo, double mc_hi, int n_mc, double fin_lo, double fin_hi, int n_fin,
                             const double* row, double* params, void* stream);
TFS_API int tfs_refine_fin(tfs_ctx* ctx, const double* params, long long n, const long long* idx, long long k,
                           int r, double d_mc, double d_fin, double* children, void* stream);

/* Number of window pixels (k_hi-k_lo+1 summed over active tranches) of each template:
 * pixel_evals = n_channels * counts[i].  counts [n] int64, host or device.  Used by the
 * benchmark for the pixel-evals/s metric and by tests for the window logic. */
TFS_API int tfs_count_pixels(tfs_ctx* ctx, const double* params, long long n, long long* counts, void* stream);

/* How tfs_eval reads the weights of the data uploaded last (C11): 0 = general per-pixel W,
 * 1 = separable W[a,m,k] = a[m] b[k] (|W - a b| <= 1e-6 a b on every pixel), 2 = separable with
 * b = 1 (weights depend on the tranche only, or weight == NULL).  -1 before the first upload. */
TFS_API int tfs_weight_structure(const tfs_ctx* ctx);

/* Templates rejected (NaN/Inf/Mc<=0) by the most recent tfs_eval on this context. */
TFS_API long long tfs_bad_param_count(const tfs_ctx* ctx);

/* Measurement hooks (bench.py).  With profiling on, the two evaluation kernels (track + gather +
 * piece sums: eval_list_kernel, which gathers from global memory, then eval_slab_kernel, which reads
 * TMA-staged shared-memory slabs) of every evaluation launch inside tfs_eval are bracketed by CUDA
 * events on the caller's stream.  tfs_get_profile_kernels synchronises those events and returns, since
 * the last call of tfs_set_profiling: the summed durations [ms] of the slab and of the list kernel, the
 * number of evaluation launches (pairs of kernels), and the number of kernels of this library launched
 * in total (all entry points).  tfs_get_profile returns the sum of the two durations.  Any output may
 * be NULL. */
TFS_API int tfs_set_profiling(tfs_ctx* ctx, int on);
TFS_API int tfs_get_profile(tfs_ctx* ctx, double* main_kernel_ms, long long* main_kernel_launches,
                            long long* kernel_launches);
TFS_API int tfs_get_profile_kernels(tfs_ctx* ctx, double* slab_kernel_ms, double* list_kernel_ms,
                                    long long* eval_launches, long long* kernel_launches);

/* Measurement hook (bench.py's per-tier operation count).  The evaluation kernels pick, warp by warp, one of three ways
 * to evaluate the Fresnel auxiliary functions of a window offset (tfs_kernels.cuh: FAR2 = leading asymptotic term, FAR =
 * fitted polynomials, NEAR = table) and also evaluate the padding slots of lanes whose tranche is inactive or whose
 * window is shorter than the warp's longest.  While the census is on, every evaluation call on the context adds the
 * number of pixel slots (lane x window offset, both channels of the pair together) it evaluated per tier to five
 * device counters:  counts[0..2] = slab kernel FAR2, FAR, NEAR;  counts[3..4] = list kernel FAR, NEAR.
 * tfs_tier_census synchronises the device, returns the counters accumulated since its previous call (counts may be NULL),
 * zeroes them and switches the census on or off.  Off by default; while on, a counting build of the two kernels runs
 * (a few atomics per work item; the default build carries no counting code), so switch it off before timing.  Counted
 * for basis 0, fresnel_mode 0, tukey_alpha 0 only (other modes leave the counters untouched). */
TFS_API int tfs_tier_census(tfs_ctx* ctx, int on, long long* counts);

/* Measurement aid for the roofline (bench.py): allocate a zero-filled scratch buffer of `bytes`
 * (choose it well inside the L2, e.g. 32 MiB), read it `iters` times with coalesced 16-byte loads from
 * one 1024-thread CTA per SM, and return the sustained read bandwidth in GB/s (CUDA events around the
 * launch; one warm-up launch first).  Synchronises `stream`.  The buffer is freed before returning. */
TFS_API int tfs_probe_l2_bandwidth(tfs_ctx* ctx, long long bytes, int iters, double* gb_per_s, void* stream);

/* Measurement aid for the roofline's arithmetic term (bench.py): how many FP32 fused multiply-add WARP instructions one
 * SM issues per clock when nothing else is in the way -- 32 resident warps per SM, 8 independent dependent chains per
 * thread, `iters` steps per chain -- for scalar FFMA (*scalar_ipc) and for the packed fma.rn.f32x2 the pixel loops use
 * (*packed_ipc; one such instruction is two fused multiply-adds per lane).  Cycles come from the SM's clock64 (median
 * over the SMs), so the figures do not depend on the clock the GPU happens to run at.  FMA-pipe lane-slots per clock per
 * SM = max(32 * scalar_ipc, 64 * packed_ipc).  Allocates and frees two small buffers; synchronises `stream`. */
TFS_API int tfs_probe_fp32_issue(tfs_ctx* ctx, int iters, double* scalar_ipc, double* packed_ipc, void* stream);

TFS_API void tfs_destroy(tfs_ctx* ctx);

/* Message of the last failure on this context (or of the last failed tfs_create when ctx is
 * NULL); never NULL; valid until the next failing call. */
TFS_API const char* tfs_last_error(const tfs_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* TFS_H */
