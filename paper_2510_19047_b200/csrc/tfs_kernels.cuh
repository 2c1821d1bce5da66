// tfs_kernels.cuh -- device code of libtfs (sm_100a).  See include/tfs.h for the operation and
// DESIGN.md section 6 for the kernel design.  Citations: P:<line> of PAPER.md, C<n> = DESIGN.md.
//
// Work decomposition (v10).  A WORK ITEM is one (template, time tile) pair; a time tile is a run of kTS
// consecutive VALID (non-gap) tranches, whatever N_seg is.  The grid is stored time-contiguous over the
// COMPACTED list of valid tranches ([k][i], i = index in that list), so a tile is a contiguous block of
// columns.  Segment boundaries cut a tile into PIECES; one warp evaluates one item and writes one partial
// per piece.  Inside an item lanes are tranches (32 at a time): fp64 0PN track per lane, then each lane
// walks its own frequency window.
//
// A pre-pass (prep_*_kernel) sorts the items of a batch into BUCKETS: per tile, by the frequency band
// (kBandStride rows) that holds the bottom of the template's track in that tile.  Items whose whole
// window fits a slab of kSlabRows rows go through eval_slab_kernel: a persistent CTA per SM claims a
// UNIT (<= kUnitItems items of one bucket), TMA (cp.async.bulk.tensor) stages the band's data slab
// [rows][kTS columns] in shared memory behind an mbarrier (two stages), and its 32 warps take the unit's
// items one by one, reading pixels with conflict-free LDS.128.  The other items (tracks that sweep many
// rows in one tile, templates that merge inside the tile) go through eval_list_kernel, which gathers
// from global memory (L2) with software-pipelined LDG.128 -- the v9 pixel loop.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace tfs {

#ifndef TFS_TS
#define TFS_TS 64
#endif
constexpr int kTS = TFS_TS;               // valid tranches per time tile (= columns of a slab); multiple of 32
static_assert(kTS == 64, "the slab kernel evaluates the two 32-tranche chunks of a tile in the two halves of packed registers");
#ifndef TFS_SLAB_ROWS
#define TFS_SLAB_ROWS 96
#endif
#ifndef TFS_SLAB_ROWS_GENERAL
#define TFS_SLAB_ROWS_GENERAL 64
#endif
#ifndef TFS_BAND_STRIDE
#define TFS_BAND_STRIDE 16
#endif
constexpr int kBandStride = TFS_BAND_STRIDE;   // rows between the bottoms of consecutive bands (even: the b table is copied from row0)
constexpr int kUnitItems = 1024;          // items per unit of the slab kernel (32 per warp)
constexpr int kListUnitItems = 32;        // items per (warp-claimed) unit of the list kernel
#ifndef TFS_WARPS
#define TFS_WARPS 32
#endif
constexpr int kWarpsPerCta = TFS_WARPS;   // list / WDM kernels: one persistent CTA of 32 warps per SM (64 registers)
#ifndef TFS_SLAB_WARPS
#define TFS_SLAB_WARPS TFS_WARPS
#endif
constexpr int kSlabWarps = TFS_SLAB_WARPS;   // slab kernel: warps of its persistent CTA (registers per thread = 65536 / (32 kSlabWarps))
constexpr int kLutN = 512;                // LUT intervals in t = 1/(1+v)
constexpr double kMtsun = 4.925490947e-6; // G Msun / c^3 [s]
constexpr double kPi = 3.14159265358979323846;
constexpr int kPadRows = 16;              // rows of zero padding behind the grid and the weights

// Weight modes (chosen by tfs_upload_data, C11):
//   kWGeneral    per-pixel weights W[alpha,m,k], read next to every data pixel
//   kWSeparable  W[alpha,m,k] = a_alpha[m] b_alpha[k]: b from a small [Nf] table, a applied once per tranche
//   kWTimeOnly   b = 1: no weight is read in the pixel loop, q' = sum |h'|^2 for both channels
constexpr int kWGeneral = 0, kWSeparable = 1, kWTimeOnly = 2;
__host__ __device__ constexpr int slab_rows(int wmode) { return wmode == kWGeneral ? TFS_SLAB_ROWS_GENERAL : TFS_SLAB_ROWS; }
constexpr int kSlabRowsMax = TFS_SLAB_ROWS > TFS_SLAB_ROWS_GENERAL ? TFS_SLAB_ROWS : TFS_SLAB_ROWS_GENERAL;
static_assert(TFS_SLAB_ROWS <= 256 && TFS_SLAB_ROWS_GENERAL <= 256, "TMA box <= 256 rows");
static_assert(kBandStride % 2 == 0 && TFS_SLAB_ROWS > kBandStride && TFS_SLAB_ROWS_GENERAL > kBandStride, "a slab must overlap the next band");

// f(v) = w (F0 + F1 w^4 + F2 w^8), g(v) = w^3 (G0 + G1 w^4 + G2 w^8), w = 1/v, valid for |v| >= kVFar
struct FarCoef {
  float F0, F1, F2, G0, G1, G2;
  float win_ell, win_b;     // window-aware template (MODE 2): taper length l = alpha/2 and shift b = 1/alpha (tfs_opts.tukey_alpha)
};

// Per-template constants, written once per batch by prep_consts_kernel (a1).
struct __align__(16) TplConst {
  double tc, phic_turns, inv5M;
  double xcoefDT;        // DT / (8 pi M):           x = f DT = X^{-3/8} xcoefDT
  double ccoef;          // (3/8) DT / (5M):         c = fdot DT^2 = x ccoef / X
  float acoef;           // amp (8 pi M)^{-2/3}:     A_m = acoef X^{-1/4}
  int ok;
  float T0r, T0i, T1r, T1i;   // constant transfer factors of the two channels of the pair (Eq. 29, C5)
};
static_assert(sizeof(TplConst) == 64, "TplConst layout");

struct Unit { int tile; int row0; unsigned off; int cnt; };   // items list[off .. off+cnt) of one bucket; cnt < 0: end marker

struct EvalArgs {
  const float4* __restrict__ grid;     // [Nf+pad][ncol] (time-contiguous over valid tranches) {Y_0.re, Y_1.re, Y_0.im, Y_1.im}, Y = W*D
  const float2* __restrict__ wgt;      // [Nf+pad][ncol] {W_0, W_1}
  const float2* __restrict__ wa;       // [ncol] {a_0, a_1} by valid-tranche index (separable weights: W = a[i] b[k])
  const float2* __restrict__ wb;       // [Nf + kPadRows + kSlabRowsMax] {b_0, b_1}
  const uint8_t* __restrict__ gap;     // [Nt] 1 = valid
  const int* __restrict__ vprefix;     // [Nt+1] number of valid tranches before m
  const int* __restrict__ valid_m;     // [ncol] the valid tranche indices, ascending (padded with the last one)
  const int* __restrict__ tile_first;  // [n_tiles+1] first piece of each tile (pieces are numbered in time order)
  const int* __restrict__ piece_end;   // [n_pieces] entry of valid_m where the piece ends (exclusive)
  const float4* __restrict__ lut;      // [kLutN+1] {a_G, a_F, b_G, b_F} (see fresnel_aux)
  const double* __restrict__ params;   // [n][8] (prep only)
  TplConst* __restrict__ tconst;       // [n]
  uint16_t* __restrict__ keys;         // [n_tiles][n] bucket of every item: 0 = no active tranche, 1 = list kernel, 2+b = band b
  unsigned* __restrict__ counts;       // [n_tiles][n_keys] items per bucket; then (scatter) the cursor of each bucket
  unsigned* __restrict__ bucket_off;   // [n_tiles][n_keys] start of each bucket in `list`
  unsigned* __restrict__ list;         // template indices, bucket by bucket (tile-major)
  Unit* __restrict__ units_slab;       // units of the slab kernel
  Unit* __restrict__ units_list;       // units of the list kernel
  int* __restrict__ n_units;           // [2] {slab, list}
  float4* __restrict__ partials;       // [n_pieces][n] {z.re, z.im, hh, 0}
  unsigned long long* bad_count;       // templates rejected
  unsigned long long* census;          // NULL (default), or [5] pixel slots evaluated per tier: slab FAR2, FAR, NEAR; list FAR, NEAR (tfs_tier_census)
  unsigned long long* work_counter;    // [2] next unclaimed unit of {slab kernel, list kernel} (zeroed before each launch)
  // optional per-template transfer table (Eq. 29, "computed once per tranche"): T_alpha(f) at n_knots
  // knots f_knot0 + j f_knot_step, linear in between, clamped outside; [n][tt_C][tt_K] complex
  const float2* __restrict__ ttab;
  int tt_K, tt_C, tt_ch0;              // knots, channels in the table, first channel of this pair
  float tt_scale, tt_off;              // knot position of bin x: x * tt_scale - tt_off
  int basis;                           // 0: complex short-time Fourier tranches (the paper); 1: real WDM wavelet pixels (tfs_wdm.cuh)
  int wdm_Hw;                          // WDM layer window half width
  double wdm_DTpix;                    // WDM pixel duration Nf dt (DT above is then 2 Nf dt = 1/DF)
  int accumulate;                      // 1: add to the partials instead of overwriting them (second channel pair)
  int t_col;                           // params columns of the pair's first transfer factor (3: T_A, T_E)
  double t3_re, t3_im;                 // t_col < 0 (the pair of channel 2, no table): the context's constant T_T (tfs_set_third_channel_factor)
  int n_ch_pair;                       // channels in this pair (1 or 2)
  long long n;                         // templates in this launch
  int Nt, Nf, ncol;
  int n_valid, n_tiles, n_keys;        // valid tranches, ceil(n_valid / kTS) (>= 1), bands + 2
  int H, adaptive;
  int slab_ok;                         // 0: every active item goes to the list kernel (fresnel_mode 1, absurd shapes)
  int wmode;
  double DT;
  double x_lo, x_hi;                   // band in bins: f_lo*DT, f_hi*DT
  double c_max;
  FarCoef far;                         // far-zone polynomials of f, g (fitted at tfs_create)
};

// a1: per-template constants from the parameter row (fp64)
__device__ __forceinline__ TplConst load_template(const double* __restrict__ p, double DT, int t_col, int n_ch) {
  TplConst t;
  const double Mc = p[0];
  t.tc = p[1];
  const double phic = p[2];
  const double amp = p[7];
  double T[4] = {0.0, 0.0, 0.0, 0.0};
  bool ok = isfinite(Mc) && isfinite(t.tc) && isfinite(phic) && isfinite(amp) && (Mc > 0.0);
#pragma unroll
  for (int c = 3; c < 7; ++c) ok = ok && isfinite(p[c]);          // a bad row is bad for every channel pair
  if (t_col >= 0) {
    T[0] = p[t_col]; T[1] = p[t_col + 1];
    if (n_ch > 1) { T[2] = p[t_col + 2]; T[3] = p[t_col + 3]; }
  }
  const double M = (ok ? Mc : 1.0) * kMtsun;
  t.inv5M = 1.0 / (5.0 * M);
  const double xcoef = 1.0 / (8.0 * kPi * M);                // f = X^{-3/8} xcoef
  t.xcoefDT = xcoef * DT;
  t.ccoef = 0.375 * DT * t.inv5M;
  // A_m = amp f^{2/3} = amp xcoef^{2/3} X^{-1/4}; a common factor of the template (fp32 is enough)
  const float cx = cbrtf((float)xcoef);
  t.acoef = (float)(ok ? amp : 0.0) * cx * cx;
  t.phic_turns = (ok ? phic : 0.0) * (0.5 / kPi);
  t.ok = ok ? 1 : 0;
  t.T0r = ok ? (float)T[0] : 0.f; t.T0i = ok ? (float)T[1] : 0.f;
  t.T1r = ok ? (float)T[2] : 0.f; t.T1i = ok ? (float)T[3] : 0.f;
  if (!ok) t.tc = 0.0;
  return t;
}

// MUFU approximations without the denormal fix-up code (inputs here are never subnormal)
__device__ __forceinline__ float rsqrt_approx(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float lg2_approx(float x) {
  float r;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float ex2_approx(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// Track point of one tranche (Eqs. 12-15 at the tranche start, C6; 0PN, C5).
struct TrackPoint {
  double x;        // f_m * DT  (position in bins)
  double c;        // fdot_m * DT^2 (bins swept in the tranche)
  double X58;      // X^{5/8}: phi_m = phic - 2 X^{5/8}
  float Xm14;      // X^{-1/4}: A_m = acoef * X^{-1/4}
  bool active;
};

// All fractional powers of X come from y = X^{-1/8}: an fp32 seed y0 = 2^{-log2(X)/8} (two MUFU ops,
// relative error d ~ 4e-7) corrected in fp64 by the binomial series of (1 - e)^{-1/8}, e = 1 - X y0^8
// ~ 8 d, to third order: the remainder is ~0.04 e^4 < 1e-20, i.e. y is exact to fp64 rounding.
// `pre` = the tranche may be active at all (valid lane, tau > DT); the band tests are applied here.
// tnow = time of the expansion point; the point can be active when tau = tc - tnow > tau_min; band test
// x >= x_lo, x + band_c c <= x_hi, c <= c_max
__device__ __forceinline__ TrackPoint track_point_at(const TplConst& t, double tnow, double tau_min,
                                                     double x_lo, double x_hi, double c_max, double band_c, bool valid) {
  TrackPoint r;
  const double tau = t.tc - tnow;
  bool act = valid && (tau > tau_min);
  const double X = act ? tau * t.inv5M : 1.0;
  double y0 = (double)ex2_approx(-0.125f * lg2_approx((float)X));
  // X outside the fp32 range (absurd masses): fall back to the seed 1/sqrt(sqrt(sqrt(X)))
  if (!(X > 1e-30 && X < 1e30)) y0 = rsqrt(sqrt(sqrt(X)));
  const double p2 = y0 * y0, p4 = p2 * p2;
  const double e = fma(-X, p4 * p4, 1.0);
  const double y = fma(y0, e * fma(e, fma(e, 51.0 / 1024.0, 9.0 / 128.0), 0.125), y0);   // X^{-1/8}
  const double y2 = y * y;                 // X^{-1/4}
  const double y3 = y2 * y;                // X^{-3/8}
  const double y4 = y2 * y2;
  r.X58 = X * y3;
  r.Xm14 = (float)y2;
  r.x = y3 * t.xcoefDT;
  r.c = r.x * t.ccoef * (y4 * y4);         // 3 f DT^2 / (8 tau), 1/tau = y^8 / (5M)
  act = act && (r.x >= x_lo) && (r.x + band_c * r.c <= x_hi) && (r.c <= c_max);
  r.active = act;
  return r;
}

__device__ __forceinline__ TrackPoint track_point(const TplConst& t, int m, double DT,
                                                  double x_lo, double x_hi, double c_max, bool valid) {
  return track_point_at(t, (double)m * DT, DT, x_lo, x_hi, c_max, 1.0, valid);
}

__device__ __forceinline__ void window(const TrackPoint& tp, int H, int adaptive, int Nf,
                                       int& k_lo, int& k_hi) {
  const int kc = (int)ceil(tp.x);                                       // C3
  const int ke = adaptive ? (int)ceil(tp.x + tp.c) : kc;                // C4
  k_lo = max(kc - H, 1);
  k_hi = min(ke + H, Nf - 1);
  k_lo = min(k_lo, Nf - 1);
  k_hi = max(k_hi, 1);
}

// LUT of the Fresnel auxiliary functions f(v), g(v) (P:184-207 defines them through Eqs. 25-26;
// A&S 7.3.5-6), tabulated against t = 1/(1+|v|) in (0, 1] with kLutN intervals:
//   entry i = {a_G, a_F, b_G, b_F}: for t within half a step of i/kLutN,
//     f(v) = t (a_F + b_F t),  g(v) = t (a_G + b_G t)
//   (the linear interpolant of F = f/t, G = g/t around node i with central-difference slope,
//    rewritten as intercept + slope*t so the fractional index is never formed).
// In shared memory it is stored LC times, copy r of entry i at 16-byte slot (i*LC + r), and lane l reads
// copy l & (LC-1): with LC = 8 the 8 lanes of a quarter-warp always hit 8 different bank groups, so an
// LDS.128 is conflict-free whatever the indices are (the slab kernel keeps 4 copies to leave room for
// its data slabs: at most 2-way conflicts).
constexpr float kMagic = 12582912.0f;          // 1.5 * 2^23: (p + kMagic) rounds p to an integer in the mantissa
constexpr unsigned kMagicBits = 0x4B400000u;

__device__ __forceinline__ float rcp_approx(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

__device__ __forceinline__ float4 lds128(unsigned addr) {
  float4 r;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "r"(addr));
  return r;
}
__device__ __forceinline__ float2 lds64(unsigned addr) {
  float2 r;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(r.x), "=f"(r.y) : "r"(addr));
  return r;
}
// LUT read: the table is written once before any read, so this one need not be volatile
__device__ __forceinline__ float4 lds128_const(unsigned addr) {
  float4 r;
  asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "r"(addr));
  return r;
}

// ----- packed fp32 pairs (sm_100a FFMA2 / FMUL2 / FADD2: two fp32 operations per issue slot) -----
// A pair lives in a 64-bit register pair {lo, hi}.  ptxas folds pk(a, a) into a broadcast operand and
// pk(-b, a) into swap / per-half negate modifiers, so these cost no extra instructions.
typedef unsigned long long f2_t;
__device__ __forceinline__ f2_t pk(float lo, float hi) {
  f2_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void upk(f2_t r, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(r));
}
__device__ __forceinline__ f2_t ffma2(f2_t a, f2_t b, f2_t c) {
  f2_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ f2_t fmul2(f2_t a, f2_t b) {
  f2_t d;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ f2_t fadd2(f2_t a, f2_t b) {
  f2_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}

// Returns GF = {g(|v|)/t, f(|v|)/t} and ts = sign(v) t, so that Godd(v) = ts GF as a complex {re, im} pair.
// lut_lane = shared address of this lane's LUT copy minus kMagicBits * (16 * LC)  (mod 2^32).
template <int MODE, int LC>
__device__ __forceinline__ void fresnel_aux(float v, unsigned lut_lane, f2_t& GF, float& ts) {
  const float a = fabsf(v);
  if (MODE != 1) {
    const float t = rcp_approx(1.0f + a);         // MUFU.RCP
    const float q = fmaf(t, (float)kLutN, kMagic);
    const float4 e = lds128_const(__float_as_uint(q) * (16u * LC) + lut_lane);   // {a_G, a_F, b_G, b_F}
    ts = copysignf(t, v);
    GF = ffma2(pk(t, t), pk(e.z, e.w), pk(e.x, e.y));
  } else {
    // the paper's Eqs. 27-28 (|v| <= 6) and the plain asymptote f = 1/(pi v), g = 0 (Eqs. 23-24, |v| > 6)
    float f, g;
    if (a > 6.0f) {
      f = __fdividef(0.318309886183790672f, a);
      g = 0.0f;
    } else {
      f = __fdividef(1.0f + 0.926f * a, 2.0f + a * (1.792f + 3.104f * a));
      g = __fdividef(1.0f, 2.0f + a * (4.142f + a * (3.492f + 6.670f * a)));
    }
    ts = copysignf(1.0f, v);
    GF = pk(g, f);
  }
}

// One pixel of one tranche (a3-a5).  The template coefficient is h = P h', P = A/sqrt(2c) exp(i phi_m)
// constant over the tranche, and (auxiliary-function form of Eq. 16)
//   h' = Godd(v0) - Godd(v1) E  [+ (1+i) exp(-i pi u^2/c) inside the swept band],
//   Godd(v) = sign(v) (g(|v|) + i f(|v|)),  E = exp(i psi), psi = pi c + 2 pi frac(x).
// The loop accumulates z'_alpha += conj(Y_alpha) h', q'_alpha += W_alpha |h'|^2 and the factor P
// (|P|^2 for q) is applied once per tranche.
//
// Three evaluations of Godd:
//   FAR  (|v0|, |v1| >= kVFar):  f(v) = w Pf(w^4), g(v) = w^3 Pg(w^4), w = 1/v, Pf and Pg quadratics
//         fitted at tfs_create (they are the asymptotic series of A&S 7.3.27-28 re-fitted on the
//         interval; odd in v, so the sign comes for free).  No table read: 2 MUFU.RCP + 10 packed ops.
//   FAR2 (|v0|, |v1| >= kVFar2): the leading terms alone, f = w/pi, g = w^3/pi^2: the next terms are
//         3/(pi^2 v^4) (< 1e-6 for v >= 24) of f and 15/(pi^2 v^4) of g (itself < 6e-4 f).  4 packed ops.
//   NEAR (anything else): the shared-memory LUT in t = 1/(1+|v|) (fresnel_aux).
// For the slow chirps that make up the bulk of every bank (|v| = sqrt(2/c) |u|) the far zones cover all
// but the ~2 pixels next to the track, and FAR2 more than half of the window.
constexpr float kVFar = 3.0f;
#ifndef TFS_VFAR2
#define TFS_VFAR2 24.0f
#endif
constexpr float kVFar2 = TFS_VFAR2;
constexpr float kNearSeries = 0.3f;    // pixel_near: midpoint expansion of F(v1) - F(v0) when pi |vm| (v1 - v0)/2 is below this

struct LaneTrack {      // per-lane (= per-tranche) constants of the pixel loop
  float sc;             // sqrt(2/c)
  float kap;            // sqrt(c/2) = 1/sc
  float c;              // v1 - v0 = sc * c
  float hc;             // 1/(2c): pi u^2/c = 2 pi (u^2 hc)
  float Er, Ei;         // exp(i psi)
};

struct LaneSums { f2_t zr, zi, q; };     // {channel 0, channel 1} pairs: Re z', Im z', q'

// grid pixel Y = {Y_0.re, Y_1.re, Y_0.im, Y_1.im}, weights Wt = {W_0, W_1} (or {b_0, b_1})
template <int WMODE>
__device__ __forceinline__ void mac(LaneSums& s, const float4 Y, const float2 Wt, float hr, float hi) {
  const f2_t Yre = pk(Y.x, Y.y), Yim = pk(Y.z, Y.w);
  s.zr = ffma2(Yre, pk(hr, hr), s.zr);            // Re conj(Y) h = Y.re hr + Y.im hi
  s.zr = ffma2(Yim, pk(hi, hi), s.zr);
  s.zi = ffma2(Yre, pk(hi, hi), s.zi);            // Im conj(Y) h = Y.re hi - Y.im hr
  s.zi = ffma2(Yim, pk(-hr, -hr), s.zi);
  if (WMODE == kWTimeOnly) {
    s.q = ffma2(pk(hr, hi), pk(hr, hi), s.q);     // {sum hr^2, sum hi^2}
  } else {
    const float h2 = fmaf(hr, hr, hi * hi);
    s.q = ffma2(pk(Wt.x, Wt.y), pk(h2, h2), s.q);
  }
}

// u = x - k; u + c is formed here, per pixel, so that it is rounded at the magnitude of u (next to the
// track, where h' is sensitive to v1 - v0, u is small).  MASKED: msk = 0 kills the contribution of a lane
// past its window.
template <int MASKED>
__device__ __forceinline__ void pixel_far(const LaneTrack& L, const FarCoef& C, float u, float msk,
                                          float& hr, float& hi) {
  const f2_t r = pk(rcp_approx(u), rcp_approx(u + L.c));
  const float kap = MASKED ? L.kap * msk : L.kap;
  const f2_t w = fmul2(r, pk(kap, kap));                         // {1/v0, 1/v1}
  const f2_t s1 = fmul2(w, w);
  const f2_t s2 = fmul2(s1, s1);
  const f2_t Pf = ffma2(s2, ffma2(s2, pk(C.F2, C.F2), pk(C.F1, C.F1)), pk(C.F0, C.F0));
  const f2_t Pg = ffma2(s2, ffma2(s2, pk(C.G2, C.G2), pk(C.G1, C.G1)), pk(C.G0, C.G0));
  const f2_t fv = fmul2(w, Pf);
  const f2_t gv = fmul2(fmul2(w, s1), Pg);
  float f0, f1, g0, g1;
  upk(fv, f0, f1);
  upk(gv, g0, g1);
  hr = fmaf(-L.Er, g1, fmaf(L.Ei, f1, g0));          // Godd(v0) - E Godd(v1)
  hi = fmaf(-L.Er, f1, fmaf(-L.Ei, g1, f0));
}

// FAR2: f = F0 w, g = G0 w^3 = (G0 / F0^3) f^3
constexpr float kG0overF03 = 3.14159265358979f;      // (1/pi^2) / (1/pi)^3 = pi
template <int MASKED>
__device__ __forceinline__ void pixel_far2(const LaneTrack& L, float u, float msk, float& hr, float& hi) {
  const f2_t r = pk(rcp_approx(u), rcp_approx(u + L.c));
  const float kf = (MASKED ? L.kap * msk : L.kap) * 0.318309886183790672f;
  const f2_t fv = fmul2(r, pk(kf, kf));                          // {f(v0), f(v1)}
  const f2_t gv = fmul2(fmul2(fv, pk(kG0overF03, kG0overF03)), fmul2(fv, fv));
  float f0, f1, g0, g1;
  upk(fv, f0, f1);
  upk(gv, g0, g1);
  hr = fmaf(-L.Er, g1, fmaf(L.Ei, f1, g0));
  hi = fmaf(-L.Er, f1, fmaf(-L.Ei, g1, f0));
}

template <int MODE, int MASKED, int LC>
__device__ __forceinline__ void pixel_near(const LaneTrack& L, float u, float msk, unsigned lut_lane,
                                           float& hr, float& hi) {
  const float v0 = L.sc * u;
  const float v1 = fmaf(L.sc, L.c, v0);
  f2_t GF0, GF1;
  float t0, t1;
  fresnel_aux<MODE, LC>(v0, lut_lane, GF0, t0);
  fresnel_aux<MODE, LC>(v1, lut_lane, GF1, t1);
  if (MASKED) { t0 *= msk; t1 *= msk; }
  const f2_t Z0 = fmul2(pk(t0, t0), GF0);                        // Godd(v0) = {re, im}
  const f2_t Z1 = fmul2(pk(t1, t1), GF1);
  float z1r, z1i;
  upk(Z1, z1r, z1i);
  f2_t h = ffma2(pk(-L.Er, -L.Er), Z1, Z0);                      // Z0 - E Z1
  h = ffma2(pk(L.Ei, L.Ei), pk(z1i, -z1r), h);
  upk(h, hr, hi);
  if (v0 < 0.0f && v1 > 0.0f) {
    // pixel inside the swept band: + (1+i) exp(-i pi u^2/c)
    float turns = u * u * L.hc;
    turns -= floorf(turns);
    float st, ct;
    __sincosf(6.283185307179586f * (turns - 0.5f), &st, &ct);        // = -(sin, cos)(2 pi turns)
    const float m = MASKED ? msk : 1.0f;
    hr -= m * (ct + st);
    hi -= m * (ct - st);
  }
  const float hs = 0.5f * L.sc * L.c;                 // (v1 - v0)/2 = sqrt(c/2)
  const float al = 3.14159265358979f * (v0 + hs);     // pi * midpoint
  if (MODE != 1 && fabsf(al) * hs < kNearSeries && hs < 0.1f) {
    // slow chirp next to the track: h' = exp(-i pi u^2/c) [F(v1) - F(v0)] is O(sqrt(2c)) while the terms above are
    // O(1) (table error 2e-7 absolute, i.e. 2e-7/sqrt(2c) relative).  Expand the integral about the midpoint vm:
    //   F(v1) - F(v0) = exp(i pi vm^2/2) int_{-h}^{h} exp(i (alpha t + beta t^2)) dt,  alpha = pi vm, beta = pi/2,
    // the prefactor's phase cancels against -pi u^2/c up to pi (u + c/4), and the integral is, to O((alpha h)^6),
    //   2h [1 + (i beta - alpha^2/2) h^2/3 + (alpha^4/24 - beta^2/2 - i alpha^2 beta/2) h^4/5]
    const float A2 = al * al, h2 = hs * hs;
    const float R = fmaf(h2 * h2, 0.2f * fmaf(A2 * A2, 1.0f / 24.0f, -1.2337006f), fmaf(A2 * h2, -1.0f / 6.0f, 1.0f));
    const float I = h2 * fmaf(h2, -0.15707963f * A2, 0.52359878f);
    float st, ct;
    __sincosf(3.14159265358979f * fmaf(0.25f, L.c, u), &st, &ct);
    const float m = 2.0f * hs * (MASKED ? msk : 1.0f);
    hr = m * fmaf(R, ct, -I * st);
    hi = m * fmaf(R, st, I * ct);
  }
}

// ------------------------------------------------------------------------------------------
// Window-aware template (MODE 2; tfs_opts.tukey_alpha > 0).  The data tranche was multiplied
// by a Tukey window before its Fourier transform, so the template pixel is Eq. 16's integrand
// times the window w(s) = 1 - [taper deficits]: with l = alpha/2, b = 1/alpha the deficits are
// [1 + cos(2 pi b s)]/2 on [0, l] and its mirror image on [1 - l, 1], and a cosine shifts u by +-b.  In the
// normalisation of h' (h = P h'):
//     h'_w = h' - Lam(u) - E Lam(-(u + c)),        Lam(w) = J(w)/2 + J(w + b)/4 + J(w - b)/4,
//     J(w) = sqrt(2c) int_0^l exp{i (2 pi w s + pi c s^2)} ds
//          = Godd(sc w) - Godd(sc (w + c l)) rho(w)  [+ (1+i) exp(-i pi w^2/c) if -c l < w < 0],
//     rho(w) = exp{i (2 pi w l + pi c l^2)},  rho(w +- b) = -rho(w)  (2 b l = 1),  sc = sqrt(2/c),
// the right taper being the left one seen from the tranche's end (s -> 1 - s turns u into -(u + c) and brings
// out the factor E = exp{i (2 pi u + pi c)}).  The taper terms are <= alpha/4 of the main pixel, so the LUT
// (absolute error 2e-7) serves every Godd here whatever |v| is.
// ------------------------------------------------------------------------------------------
template <int LC>
__device__ __forceinline__ void godd_lut(float v, unsigned lut_lane, float& gr, float& gi) {
  f2_t GF;
  float ts;
  fresnel_aux<0, LC>(v, lut_lane, GF, ts);
  upk(fmul2(pk(ts, ts), GF), gr, gi);
}

template <int LC>
__device__ __forceinline__ void taper_J(const LaneTrack& L, float w, float cl, float rr, float ri, unsigned lut_lane,
                                        float& jr, float& ji) {
  float a0r, a0i, a1r, a1i;
  godd_lut<LC>(L.sc * w, lut_lane, a0r, a0i);
  godd_lut<LC>(L.sc * (w + cl), lut_lane, a1r, a1i);
  jr = a0r - fmaf(a1r, rr, -a1i * ri);
  ji = a0i - fmaf(a1r, ri, a1i * rr);
  if (w < 0.0f && w + cl > 0.0f) {
    // the stationary point lies inside the taper: + (1+i) exp(-i pi w^2/c), pi w^2/c < pi c l^2
    float st, ct;
    __sincosf(6.283185307179586f * (w * w * L.hc), &st, &ct);
    jr += ct + st;
    ji += ct - st;
  }
}

template <int LC>
__device__ __forceinline__ void taper_lambda(const LaneTrack& L, float w, float ell, float b, unsigned lut_lane,
                                             float& lr, float& li) {
  const float cl = L.c * ell;
  float turns = fmaf(w, ell, 0.5f * cl * ell);         // (2 pi w l + pi c l^2) / 2 pi
  turns -= floorf(turns);
  float sr, cr;
  __sincosf(6.283185307179586f * (turns - 0.5f), &sr, &cr);     // = -(sin, cos)(2 pi turns)
  float j0r, j0i, jpr, jpi, jmr, jmi;
  taper_J<LC>(L, w, cl, -cr, -sr, lut_lane, j0r, j0i);
  taper_J<LC>(L, w + b, cl, cr, sr, lut_lane, jpr, jpi);        // rho(w +- b) = -rho(w)
  taper_J<LC>(L, w - b, cl, cr, sr, lut_lane, jmr, jmi);
  lr = fmaf(0.25f, jpr + jmr, 0.5f * j0r);
  li = fmaf(0.25f, jpi + jmi, 0.5f * j0i);
}

// h' -> h'_w for the pixel at u (msk = 0 for a lane past its window)
template <int LC>
__device__ __forceinline__ void taper_terms(const LaneTrack& L, const FarCoef& C, float u, float msk, unsigned lut_lane,
                                            float& hr, float& hi) {
  float l0r, l0i, l1r, l1i;
  taper_lambda<LC>(L, u, C.win_ell, C.win_b, lut_lane, l0r, l0i);
  taper_lambda<LC>(L, -(u + L.c), C.win_ell, C.win_b, lut_lane, l1r, l1i);
  hr -= msk * (l0r + fmaf(L.Er, l1r, -L.Ei * l1i));
  hi -= msk * (l0i + fmaf(L.Er, l1i, L.Ei * l1r));
}

constexpr int kZNear = 0, kZFar = 1, kZFar2 = 2;

// one pixel of kind KIND at offset jj (u = x - k of that pixel, stepped by the caller)
template <int KIND, int MODE, int WMODE, int MASKED, int LC>
__device__ __forceinline__ void pixel_kind(const LaneTrack& L, const FarCoef& C, int jj, int Wm, const float4 Yc,
                                           const float2 Wc, float u, unsigned lut_lane, LaneSums& s) {
  const float msk = (MASKED && jj >= Wm) ? 0.0f : 1.0f;
  float hr, hi;
  if (KIND == kZNear) pixel_near<MODE, MASKED, LC>(L, u, msk, lut_lane, hr, hi);
  else if (KIND == kZFar) pixel_far<MASKED>(L, C, u, msk, hr, hi);
  else pixel_far2<MASKED>(L, u, msk, hr, hi);
  if (MODE == 2) taper_terms<LC>(L, C, u, msk, lut_lane, hr, hi);
  mac<WMODE>(s, Yc, Wc, hr, hi);
}

// ------------------------------------------------------------------------------------------
// Pixel loop of the LIST kernel (global-memory gather).  Every lane walks its own window, offsets
// j = 0 ... Wm-1 from its k_lo, in groups of kGroup offsets.  The gather is software-pipelined through
// two register buffers: the loads of group g+1 are issued before the arithmetic of group g.  It is never
// predicated: the grid is allocated with kPadRows zeroed rows past Nf-1, so reading a few pixels past the
// end of a window stays in bounds, and an inactive lane reads pixel `idx` with stride 0 (its sums are
// multiplied by P = 0 at the end; the upload zeroes non-finite pixels, so whatever it reads is finite).
// Offsets [JA, JB) (warp-uniform) are the NEAR zone, evaluated from the LUT with the in-band test; every
// other offset is FAR for every active lane, and a group that does not touch the near zone runs
// straight-line far-zone code.  Groups that lie below Wmin (the shortest active window) need no per-lane
// test at all; the groups that reach past it multiply the contribution of lanes past their own window
// by zero.  Chunks whose windows differ by more than kRagMax pixels also clamp every load offset.
// ------------------------------------------------------------------------------------------
#ifndef TFS_GROUP
#define TFS_GROUP 2
#endif
constexpr int kGroup = TFS_GROUP;
constexpr int kRagMax = kPadRows - 2 * kGroup;   // largest Wmax - Wmin handled without clamping the loads
static_assert(kRagMax >= 1, "kPadRows too small for kGroup");
constexpr int kLutCopiesList = 8;

// ZONES: 1 = test the offset against the near zone, 0 = the offset is known to be far.
// The bin offset u = x - k is formed per pixel as fr + n with fr = x - round(x) in [-1/2, 1/2] (from the fp64 x)
// and n = round(x) - k an exact small integer: for the bin nearest the track (n = 0) u = fr exactly, elsewhere
// |u| >= 1/2 and the rounding is relative.  A value stepped down from u(k_lo) ~ H would carry 1 ulp of H against
// u ~ 1e-5 when the track sits on a bin (found by tests/test_gpu_parity.py::test_precision_worst_case_hunt).
template <int MODE, int WMODE, int MASKED, int ZONES>
__device__ __forceinline__ void pixel_step(const LaneTrack& L, const FarCoef& C, int jj, int Wm, int JA, int JB,
                                           const float4 Yc, const float2 Wc, float fr, float& nn, unsigned lut_lane,
                                           LaneSums& s) {
  const float u = fr + nn;
  if (ZONES && jj >= JA && jj < JB) pixel_kind<kZNear, MODE, WMODE, MASKED, kLutCopiesList>(L, C, jj, Wm, Yc, Wc, u, lut_lane, s);
  else pixel_kind<kZFar, MODE, WMODE, MASKED, kLutCopiesList>(L, C, jj, Wm, Yc, Wc, u, lut_lane, s);
  nn -= 1.0f;
}

struct PixelBuf { float4 Y[kGroup]; float2 W[kGroup]; };

// loads offsets j0 ... j0+kGroup-1 of the lane's window (CLAMP: not past offset jlast).
// kb = k_lo and kstp = 1 for an active lane (0, 0 otherwise): row index of the b table (kWSeparable).
template <int CLAMP, int WMODE>
__device__ __forceinline__ void load_group(const EvalArgs& a, PixelBuf& B, int idx, int stp, int kb, int kstp, int j0,
                                           int jlast) {
#pragma unroll
  for (int p = 0; p < kGroup; ++p) {
    const int jj = CLAMP ? min(j0 + p, jlast) : (j0 + p);
    const int i = idx + jj * stp;
#ifdef TFS_BOUNDS_CHECK
#ifndef TFS_BOUNDS_PAD
#define TFS_BOUNDS_PAD kPadRows   // (a smaller value makes the check fail on purpose: tests the checker)
#endif
    // debug builds only: the gather is unpredicated, so prove it stays inside the padded arrays
    if (i < 0 || i >= (a.Nf + TFS_BOUNDS_PAD) * a.ncol || kb + jj * kstp < 0 || kb + jj * kstp >= a.Nf + TFS_BOUNDS_PAD) __trap();
#endif
    B.Y[p] = __ldg(a.grid + i);
    if (WMODE == kWGeneral) B.W[p] = __ldg(a.wgt + i);
    if (WMODE == kWSeparable) B.W[p] = __ldg(a.wb + kb + jj * kstp);
  }
}

template <int MODE, int WMODE, int MASKED>
__device__ __forceinline__ void compute_group(const LaneTrack& L, const FarCoef& C, const PixelBuf& B, int j0, int Wm,
                                              int Wmax, int JA, int JB, float fr, float& nn, unsigned lut_lane, LaneSums& s) {
  if (j0 < JB && j0 + kGroup > JA) {
#pragma unroll
    for (int p = 0; p < kGroup; ++p)
      if (!MASKED || j0 + p < Wmax)
        pixel_step<MODE, WMODE, MASKED, 1>(L, C, j0 + p, Wm, JA, JB, B.Y[p], B.W[p], fr, nn, lut_lane, s);
  } else {
#pragma unroll
    for (int p = 0; p < kGroup; ++p)
      if (!MASKED || j0 + p < Wmax)
        pixel_step<MODE, WMODE, MASKED, 0>(L, C, j0 + p, Wm, JA, JB, B.Y[p], B.W[p], fr, nn, lut_lane, s);
  }
}

// one group from buffer B: unmasked while the whole group lies below Wmin
template <int MODE, int WMODE>
__device__ __forceinline__ void compute_group_auto(const LaneTrack& L, const FarCoef& C, const PixelBuf& B, int j0,
                                                   int Wm, int Wmin, int Wmax, int JA, int JB, float fr, float& nn,
                                                   unsigned lut_lane, LaneSums& s) {
  if (j0 + kGroup <= Wmin) compute_group<MODE, WMODE, 0>(L, C, B, j0, Wm, Wmax, JA, JB, fr, nn, lut_lane, s);
  else compute_group<MODE, WMODE, 1>(L, C, B, j0, Wm, Wmax, JA, JB, fr, nn, lut_lane, s);
}

// idx = pixel index of offset 0, stp = ncol for an active lane and 0 otherwise, Wm = window length (>= 1
// for active lanes, 0 otherwise)
template <int MODE, int WMODE>
__device__ __forceinline__ void pixel_loop_global(const EvalArgs& a, const LaneTrack& L, const FarCoef& C, int Wm, int Wmin,
                                                  int Wmax, int JA, int JB, int idx, int stp, int kb, int kstp, float fr,
                                                  float nn, unsigned lut_lane, LaneSums& s) {
  PixelBuf A, B;
#pragma unroll
  for (int p = 0; p < kGroup; ++p) { A.W[p] = make_float2(0.f, 0.f); B.W[p] = make_float2(0.f, 0.f); }
  const int jlast = max(Wm - 1, 0);
  if (Wmax - Wmin <= kRagMax) {
    // windows of (nearly) equal length, the usual case: nothing is clamped (the loads stay within
    // kRagMax + 2 kGroup rows of every lane's window: zeroed pad rows), only the groups that reach
    // past Wmin are masked
    load_group<0, WMODE>(a, A, idx, stp, kb, kstp, 0, jlast);
    for (int j = 0; j < Wmax; j += 2 * kGroup) {
      if (j + kGroup < Wmax) load_group<0, WMODE>(a, B, idx, stp, kb, kstp, j + kGroup, jlast);
      compute_group_auto<MODE, WMODE>(L, C, A, j, Wm, Wmin, Wmax, JA, JB, fr, nn, lut_lane, s);
      if (j + kGroup >= Wmax) break;
      if (j + 2 * kGroup < Wmax) load_group<0, WMODE>(a, A, idx, stp, kb, kstp, j + 2 * kGroup, jlast);
      compute_group_auto<MODE, WMODE>(L, C, B, j + kGroup, Wm, Wmin, Wmax, JA, JB, fr, nn, lut_lane, s);
    }
  } else {
    // very ragged chunk (wide tracks next to narrow ones): every load clamped, every step masked
    load_group<1, WMODE>(a, A, idx, stp, kb, kstp, 0, jlast);
    for (int j = 0; j < Wmax; j += 2 * kGroup) {
      load_group<1, WMODE>(a, B, idx, stp, kb, kstp, j + kGroup, jlast);
      compute_group<MODE, WMODE, 1>(L, C, A, j, Wm, Wmax, JA, JB, fr, nn, lut_lane, s);
      if (j + kGroup >= Wmax) break;
      load_group<1, WMODE>(a, A, idx, stp, kb, kstp, j + 2 * kGroup, jlast);
      compute_group<MODE, WMODE, 1>(L, C, B, j + kGroup, Wm, Wmax, JA, JB, fr, nn, lut_lane, s);
    }
  }
}

#ifndef TFS_LUT_COPIES_SLAB
#define TFS_LUT_COPIES_SLAB 4
#endif
constexpr int kLutCopiesSlab = TFS_LUT_COPIES_SLAB;

// ------------------------------------------------------------------------------------------
// One work item: template `it` on time tile `tile` (rows a2-a7).  LANES ARE TRANCHES: lane l owns the
// l-th valid (non-gap) tranche of the current chunk of 32, computes its track point in fp64 and then
// walks its own window pixel by pixel.  Per chunk the window offsets are split (warp-uniformly) into the
// NEAR zone around the track, evaluated from the shared-memory LUT, and the FAR zones, evaluated from
// asymptotic polynomials in packed fp32.  The tranche's sums are multiplied by P, combined over the two
// channels with the transfer factors (a6: constant per template, or interpolated at f_m from the
// template's table, Eq. 29) and added to the lane's running sums of the current piece; when a piece
// ends -- inside a chunk at a segment boundary, or at the end of the tile -- the lanes are summed with a
// shuffle butterfly and the piece's partial {z, hh} is stored.
// This is the item evaluator of eval_list_kernel (pixels gathered from global memory); eval_slab_kernel uses
// eval_item_pair below.
// ------------------------------------------------------------------------------------------
template <int MODE, int WMODE, bool CENSUS>
__device__ __forceinline__ void eval_item(const EvalArgs& a, const long long it, const int tile, const int lane,
                                          const unsigned lut_lane) {
  const TplConst T = a.tconst[it];
  // valid (non-gap) tranches of the tile: entries [i0, i1) of the compacted list (C10), cut by the
  // segment boundaries into pieces [p, p_stop)
  const int i0 = tile * kTS, i1 = min(i0 + kTS, a.n_valid);
  int p = a.tile_first[tile];
  const int p_stop = a.tile_first[tile + 1];
  int pend = p < p_stop ? a.piece_end[p] : i1;
  float accr = 0.f, acci = 0.f, acch = 0.f;      // this lane's running sums of the current piece

  // close piece p: sum the lanes (fp32 butterfly: 32 terms), store, reset
  auto flush = [&]() {
    float r0 = accr, r1 = acci, r2 = acch;
    accr = 0.f; acci = 0.f; acch = 0.f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      r0 += __shfl_xor_sync(0xffffffffu, r0, o);
      r1 += __shfl_xor_sync(0xffffffffu, r1, o);
      r2 += __shfl_xor_sync(0xffffffffu, r2, o);
    }
    if (lane == 0) {
      float4* dst = a.partials + (long long)p * a.n + it;
      float4 v = make_float4(r0, r1, r2, 0.f);
      if (a.accumulate) { const float4 o = *dst; v.x += o.x; v.y += o.y; v.z += o.z; }
      *dst = v;
    }
  };

  for (int ic = i0; ic < i1; ic += 32) {
    // ---------------- track point of this lane's tranche (a2) ----------------
    const int i = ic + lane;
    const bool valid = i < i1;
    const int m = a.valid_m[valid ? i : i0];
    const TrackPoint tp = track_point(T, m, a.DT, a.x_lo, a.x_hi, a.c_max, valid);
    const unsigned act_mask = __ballot_sync(0xffffffffu, tp.active);
    const int cend = min(ic + 32, i1);
    const bool closes = p < p_stop && pend <= cend;   // a piece ends inside this chunk (warp-uniform)
    float vr = 0.f, vi = 0.f, vq = 0.f;               // this tranche's contribution to z and hh
    if (act_mask != 0u) {
      int Wm = 0, k_lo = 0, ja = 0x7fffffff, jb = 0;
      float fr = 0.f, n0 = -1.f, Pr = 0.f, Pi = 0.f;       // u_j = fr + (n0 - j)
      LaneTrack L;        // inactive lanes: u_j = -1 - j, u_j + c = -0.5 - j (finite h' on finite data)
      L.sc = 1.f; L.kap = 1.f; L.c = 0.5f; L.hc = 0.f; L.Er = 0.f; L.Ei = 0.f;
      if (tp.active) {
        int k_hi;
        window(tp, a.H, a.adaptive, a.Nf, k_lo, k_hi);
        Wm = k_hi - k_lo + 1;
        const double flx = floor(tp.x);
        const int kr = __double2int_rn(tp.x);
        fr = (float)(tp.x - (double)kr);               // x - k = (x - round(x)) + (round(x) - k): see pixel_step
        n0 = (float)(kr - k_lo);
        const float u = fr + n0;
        // phases in turns, reduced in fp64 (phi reaches ~1e8 rad), then to [-1/2, 1/2)
        double tphi = T.phic_turns - tp.X58 * (1.0 / kPi);
        tphi -= floor(tphi);
        double tpsi = 0.5 * tp.c + (tp.x - flx);
        tpsi -= floor(tpsi);
        float sphi, cphi, spsi, cpsi;
        __sincosf(6.283185307179586f * ((float)tphi - 0.5f), &sphi, &cphi);     // = -(sin, cos)(2 pi tphi)
        __sincosf(6.283185307179586f * ((float)tpsi - 0.5f), &spsi, &cpsi);
        const float cf = (float)tp.c;
        L.sc = rsqrt_approx(0.5f * cf);
        L.kap = 0.5f * cf * L.sc;                                               // sqrt(c/2)
        L.c = cf;
        L.hc = 0.5f * rcp_approx(cf);
        const float pre = -(T.acoef * tp.Xm14) * (0.5f * L.sc);               // -A_m / sqrt(2c)
        Pr = pre * cphi;
        Pi = pre * sphi;
        L.Er = -cpsi;
        L.Ei = -spsi;
        // near zone of this lane: offsets j with |v0| < kVFar or |v1| < kVFar, i.e. -(c + d) < u - j < d
        const float d = fmaf(kVFar, L.kap, 1e-3f);
        ja = max(__float2int_rd(u - d) + 1, 0);
        jb = __float2int_ru(u + cf + d);
      }
      const int Wmax = __reduce_max_sync(0xffffffffu, Wm);
      const int Wmin = __reduce_min_sync(0xffffffffu, tp.active ? Wm : 0x7fffffff);
      int JA = __reduce_min_sync(0xffffffffu, ja);
      int JB = min(__reduce_max_sync(0xffffffffu, jb), Wmax);
      if (MODE == 1) { JA = 0; JB = Wmax; }          // the paper's approximants are used for every pixel
      JA = min(JA, JB);
      if (CENSUS && lane == 0) {        // measurement only: 32 pixel slots per offset, NEAR in [JA, JB)
        atomicAdd(a.census + 3, 32ull * (unsigned)(Wmax - (JB - JA)));
        atomicAdd(a.census + 4, 32ull * (unsigned)(JB - JA));
      }

      // ---------------- pixel loop (a3-a5): lane walks its own window ----------------
      LaneSums s;
      s.zr = pk(0.f, 0.f); s.zi = pk(0.f, 0.f); s.q = pk(0.f, 0.f);
      {
        const int stp = tp.active ? a.ncol : 0;
        const int idx = tp.active ? k_lo * a.ncol + i : (valid ? i : i0);
        pixel_loop_global<MODE, WMODE>(a, L, a.far, Wm, Wmin, Wmax, JA, JB, idx, stp, tp.active ? k_lo : 0,
                                       tp.active ? 1 : 0, fr, n0, lut_lane, s);
      }
      // ---------------- a6: transfer factors, the tranche's factor P, weights a[i] ----------------
      float T0r = T.T0r, T0i = T.T0i, T1r = T.T1r, T1i = T.T1i;
      if (a.ttab != nullptr) {
        // T_alpha(f_m) from the template's table: linear between knots, clamped outside (Eq. 29)
        const int K = a.tt_K;
        float sx = fmaf((float)tp.x, a.tt_scale, -a.tt_off);
        sx = fminf(fmaxf(sx, 0.f), (float)(K - 1));
        int kn = min((int)sx, max(K - 2, 0));
        const float tf = K > 1 ? sx - (float)kn : 0.f;
        const int kn1 = min(kn + 1, K - 1);
        const float2* tb = a.ttab + ((size_t)it * a.tt_C + a.tt_ch0) * K;
        const float2 A0 = __ldg(tb + kn), A1 = __ldg(tb + kn1);
        T0r = fmaf(tf, A1.x - A0.x, A0.x); T0i = fmaf(tf, A1.y - A0.y, A0.y);
        T1r = 0.f; T1i = 0.f;
        if (a.tt_ch0 + 1 < a.tt_C && a.n_ch_pair > 1) {
          const float2 B0 = __ldg(tb + K + kn), B1 = __ldg(tb + K + kn1);
          T1r = fmaf(tf, B1.x - B0.x, B0.x); T1i = fmaf(tf, B1.y - B0.y, B0.y);
        }
      }
      float zr0, zr1, zi0, zi1, q0, q1;
      upk(s.zr, zr0, zr1); upk(s.zi, zi0, zi1); upk(s.q, q0, q1);
      if (WMODE == kWTimeOnly) { q0 = q0 + q1; q1 = q0; }      // the loop summed {hr^2, hi^2}
      // z' = T_0 z'_0 + T_1 z'_1 ;  q' = |T_0|^2 a_0 q'_0 + |T_1|^2 a_1 q'_1   (Eq. 29, Eq. 31)
      const float zcr = fmaf(T0r, zr0, fmaf(-T0i, zi0, fmaf(T1r, zr1, -T1i * zi1)));
      const float zci = fmaf(T0r, zi0, fmaf(T0i, zr0, fmaf(T1r, zi1, T1i * zr1)));
      float w0 = fmaf(T0r, T0r, T0i * T0i), w1 = fmaf(T1r, T1r, T1i * T1i);
      if (WMODE != kWGeneral) {
        const float2 am = __ldg(a.wa + (valid ? i : i0));
        w0 *= am.x; w1 *= am.y;
      }
      const float P2 = fmaf(Pr, Pr, Pi * Pi);
      vr = fmaf(Pr, zcr, -Pi * zci);                  // Re (P z')
      vi = fmaf(Pr, zci, Pi * zcr);                   // Im (P z')
      vq = P2 * fmaf(w0, q0, w1 * q1);
      if (!closes) { accr += vr; acci += vi; acch += vq; }    // the usual case: the whole chunk belongs to the current piece
    }
    if (closes) {
      // every piece that ends inside this chunk (a segment boundary, or the end of the tile) takes the
      // lanes before its end and is closed; the lanes behind the last such end open the next piece
      int lo = 0;
      for (;;) {
        const bool ends = p < p_stop && pend <= cend;
        const int hi = ends ? pend - ic : 32;
        if (lane >= lo && lane < hi) { accr += vr; acci += vi; acch += vq; }
        if (!ends) break;
        flush();
        ++p;
        if (p < p_stop) pend = a.piece_end[p];
        lo = hi;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// One work item of the SLAB kernel.  A tile is kTS = 64 valid tranches = two chunks of 32, and every lane
// evaluates TWO tranches at once -- entry i0 + lane of the valid-tranche list (half 0) and entry
// i0 + 32 + lane (half 1) -- with the two tranches in the two halves of packed fp32 registers: every
// per-pixel instruction outside the polynomials (which were already packed over v0, v1) then serves two
// pixels, the loop and zone overheads are paid once for both, and the window-offset zones are taken over
// all 64 tranches.  Offsets are relative to each tranche's own k_lo, so the zones line up.
//   [0, J2A) FAR2 | [J2A, JA) FAR | [JA, JB) NEAR | [JB, J2B) FAR | [J2B, Wmin) FAR2 | [Wmin, Wmax) masked
// The data sit in shared memory as [row][kTS columns] float4 (plus [row][kTS] float2 weights, or the band's
// rows of the b table); lane l of half h reads column 32 h + l, so the 8 lanes of a quarter-warp always
// fall in 8 different 16-byte bank groups: an LDS.128 is conflict-free whatever rows the lanes are on.
// An inactive tranche walks rows row0, row0+1, ... of its own column (always inside the slab).
// ------------------------------------------------------------------------------------------
struct PairTrack {        // per-lane constants of the pixel loop, {half 0, half 1}
  f2_t kap;               // sqrt(c/2)
  f2_t kapf;              // sqrt(c/2) / pi
  f2_t c;                 // fdot DT^2
  f2_t Er, Ei;            // exp(i psi)
  f2_t sc, hc;            // near zone only: sqrt(2/c), 1/(2c)
};

struct PairSums { f2_t zr[2], zi[2], q[2]; };   // [half] {channel 0, channel 1}; kWTimeOnly: q[0] = sum hr^2, q[1] = sum hi^2 as {half 0, half 1}

template <int WMODE>
struct SlabPair {
  unsigned y[2];          // shared address of the pixel of offset 0, per half
  unsigned w[2];          // kWGeneral: same in the weight slab; kWSeparable: row of the b table
#ifdef TFS_BOUNDS_CHECK
  int row_rel[2], rows;
#endif
  __device__ __forceinline__ void load(int h, int j, float4& Y, float2& W) const {
#ifdef TFS_BOUNDS_CHECK
    if (row_rel[h] + j < 0 || row_rel[h] + j >= rows) __trap();
#endif
    Y = lds128(y[h] + (unsigned)j * (kTS * 16u));
    if (WMODE == kWGeneral) W = lds64(w[h] + (unsigned)j * (kTS * 8u));
    else if (WMODE == kWSeparable) W = lds64(w[h] + (unsigned)j * 8u);
    else W = make_float2(0.f, 0.f);
  }
};

// template coefficient h' of the pixel of offset j for both halves: hr = {hr_0, hr_1}, hi = {hi_0, hi_1}
template <int KIND, int MASKED>
__device__ __forceinline__ void pair_h(const PairTrack& L, const FarCoef& C, f2_t u, f2_t msk, unsigned lut_lane, f2_t& hr, f2_t& hi) {
  if (KIND == kZNear) {
    float u0, u1, m0 = 1.f, m1 = 1.f, hr0, hr1, hi0, hi1;
    upk(u, u0, u1);
    if (MASKED) upk(msk, m0, m1);
    LaneTrack A, B;
    upk(L.sc, A.sc, B.sc); upk(L.kap, A.kap, B.kap); upk(L.c, A.c, B.c); upk(L.hc, A.hc, B.hc);
    upk(L.Er, A.Er, B.Er); upk(L.Ei, A.Ei, B.Ei);
    pixel_near<0, MASKED, kLutCopiesSlab>(A, u0, m0, lut_lane, hr0, hi0);
    pixel_near<0, MASKED, kLutCopiesSlab>(B, u1, m1, lut_lane, hr1, hi1);
    hr = pk(hr0, hr1);
    hi = pk(hi0, hi1);
    return;
  }
  float u0, u1, c0, c1;
  const f2_t uc = fadd2(u, L.c);          // u + c, rounded at the magnitude of u
  upk(u, u0, u1);
  upk(uc, c0, c1);
  const f2_t r0 = pk(rcp_approx(u0), rcp_approx(u1));      // 1/u of both halves
  const f2_t r1 = pk(rcp_approx(c0), rcp_approx(c1));      // 1/(u + c)
  f2_t f0, f1, g0, g1;
  if (KIND == kZFar) {
    const f2_t kap = MASKED ? fmul2(L.kap, msk) : L.kap;
    const f2_t w0 = fmul2(r0, kap), w1 = fmul2(r1, kap);   // 1/v0, 1/v1
    const f2_t a0 = fmul2(w0, w0), a1 = fmul2(w1, w1);
    const f2_t b0 = fmul2(a0, a0), b1 = fmul2(a1, a1);
    const f2_t F2 = pk(C.F2, C.F2), F1 = pk(C.F1, C.F1), F0 = pk(C.F0, C.F0);
    const f2_t G2 = pk(C.G2, C.G2), G1 = pk(C.G1, C.G1), G0 = pk(C.G0, C.G0);
    f0 = fmul2(w0, ffma2(b0, ffma2(b0, F2, F1), F0));
    f1 = fmul2(w1, ffma2(b1, ffma2(b1, F2, F1), F0));
    g0 = fmul2(fmul2(w0, a0), ffma2(b0, ffma2(b0, G2, G1), G0));
    g1 = fmul2(fmul2(w1, a1), ffma2(b1, ffma2(b1, G2, G1), G0));
  } else {
    const f2_t kf = MASKED ? fmul2(L.kapf, msk) : L.kapf;
    const f2_t pi2 = pk(kG0overF03, kG0overF03);
    f0 = fmul2(r0, kf);
    f1 = fmul2(r1, kf);
    g0 = fmul2(fmul2(f0, pi2), fmul2(f0, f0));
    g1 = fmul2(fmul2(f1, pi2), fmul2(f1, f1));
  }
  const f2_t nEr = L.Er ^ 0x8000000080000000ULL, nEi = L.Ei ^ 0x8000000080000000ULL;
  hr = ffma2(nEr, g1, ffma2(L.Ei, f1, g0));            // Godd(v0) - E Godd(v1)
  hi = ffma2(nEr, f1, ffma2(nEi, g1, f0));
}

// z', q' of both halves for the pixel of offset j
template <int KIND, int WMODE, int MASKED>
__device__ __forceinline__ void pair_pixel(const SlabPair<WMODE>& sl, const PairTrack& L, const FarCoef& C, int j, f2_t u,
                                           int Wm0, int Wm1, unsigned lut_lane, PairSums& s) {
  float4 Y0, Y1;
  float2 W0, W1;
  sl.load(0, j, Y0, W0);
  sl.load(1, j, Y1, W1);
  f2_t msk = 0;
  if (MASKED) msk = pk(j < Wm0 ? 1.f : 0.f, j < Wm1 ? 1.f : 0.f);
  f2_t hr, hi;
  pair_h<KIND, MASKED>(L, C, u, msk, lut_lane, hr, hi);
  float hr0, hr1, hi0, hi1;
  upk(hr, hr0, hr1);
  upk(hi, hi0, hi1);
  {
    const f2_t Yre = pk(Y0.x, Y0.y), Yim = pk(Y0.z, Y0.w);
    s.zr[0] = ffma2(Yre, pk(hr0, hr0), s.zr[0]);
    s.zr[0] = ffma2(Yim, pk(hi0, hi0), s.zr[0]);
    s.zi[0] = ffma2(Yre, pk(hi0, hi0), s.zi[0]);
    s.zi[0] = ffma2(Yim, pk(-hr0, -hr0), s.zi[0]);
  }
  {
    const f2_t Yre = pk(Y1.x, Y1.y), Yim = pk(Y1.z, Y1.w);
    s.zr[1] = ffma2(Yre, pk(hr1, hr1), s.zr[1]);
    s.zr[1] = ffma2(Yim, pk(hi1, hi1), s.zr[1]);
    s.zi[1] = ffma2(Yre, pk(hi1, hi1), s.zi[1]);
    s.zi[1] = ffma2(Yim, pk(-hr1, -hr1), s.zi[1]);
  }
  if (WMODE == kWTimeOnly) {
    s.q[0] = ffma2(hr, hr, s.q[0]);
    s.q[1] = ffma2(hi, hi, s.q[1]);
  } else {
    float h20, h21;
    upk(ffma2(hr, hr, fmul2(hi, hi)), h20, h21);
    s.q[0] = ffma2(pk(W0.x, W0.y), pk(h20, h20), s.q[0]);
    s.q[1] = ffma2(pk(W1.x, W1.y), pk(h21, h21), s.q[1]);
  }
}

#ifndef TFS_PAIR_UNROLL
#define TFS_PAIR_UNROLL 1
#endif
constexpr int kPairUnroll = TFS_PAIR_UNROLL;

// offsets [jb, je) of kind KIND.  u = x - k is formed per pixel as fr + n, fr = x - round(x), n = round(x) - k an
// exact small integer (n0 at offset 0): the bin nearest the track gets u = fr exactly (see pixel_step).
template <int KIND, int WMODE>
__device__ __forceinline__ void pair_zone(const SlabPair<WMODE>& sl, const PairTrack& L, const FarCoef& C, int jb, int je,
                                          f2_t fr, f2_t n0, unsigned lut_lane, PairSums& s) {
  const float fj = (float)jb;
  f2_t nn = fadd2(n0, pk(-fj, -fj));             // exact: small integers
  const f2_t m1 = pk(-1.f, -1.f);
#pragma unroll(kPairUnroll)
  for (int j = jb; j < je; ++j) {
    pair_pixel<KIND, WMODE, 0>(sl, L, C, j, fadd2(fr, nn), 0, 0, lut_lane, s);
    nn = fadd2(nn, m1);
  }
}

template <int WMODE, bool CENSUS>
__device__ __forceinline__ void eval_item_pair(const EvalArgs& a, const long long it, const int tile, const int lane,
                                               const unsigned lut_lane, const unsigned slab_y, const unsigned slab_w,
                                               const int row0) {
  const int i0 = tile * kTS, i1 = min(i0 + kTS, a.n_valid);
  int p = a.tile_first[tile];
  const int p_stop = a.tile_first[tile + 1];
  int pend = p < p_stop ? a.piece_end[p] : i1;
  float accr = 0.f, acci = 0.f, acch = 0.f;      // this lane's running sums of the current piece

  // ---------------- track points of this lane's two tranches (a2) ----------------
  float frx[2], nn0[2], Pr[2], Pi[2], kap[2], cc[2], Er[2], Ei[2], sc[2], hc[2], xf[2];
  int Wm[2], krel[2], idxv[2];
  int ja = 0x7fffffff, jb = 0, j2a = 0x7fffffff, j2b = 0, wmin = 0x7fffffff;
  bool any = false;
  {
    const TplConst T = a.tconst[it];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int i = i0 + 32 * h + lane;
      const bool valid = i < i1;
      idxv[h] = valid ? i : i0;
      const int m = a.valid_m[idxv[h]];
      const TrackPoint tp = track_point(T, m, a.DT, a.x_lo, a.x_hi, a.c_max, valid);
      // an inactive tranche: u_j = -1 - j, u_j + c = -0.5 - j (finite h' on finite data), P = 0
      Wm[h] = 0; krel[h] = 0; frx[h] = 0.f; nn0[h] = -1.f; Pr[h] = 0.f; Pi[h] = 0.f; kap[h] = 1.f; cc[h] = 0.5f; Er[h] = 0.f; Ei[h] = 0.f;
      sc[h] = 1.f; hc[h] = 0.f; xf[h] = 0.f;
      if (tp.active) {
        any = true;
        int k_lo, k_hi;
        window(tp, a.H, a.adaptive, a.Nf, k_lo, k_hi);
        Wm[h] = k_hi - k_lo + 1;
        krel[h] = k_lo - row0;
        wmin = min(wmin, Wm[h]);
        const int kfl = __double2int_rd(tp.x), kr = __double2int_rn(tp.x);
        const double fr = tp.x - (double)kfl;
        frx[h] = (float)(tp.x - (double)kr);               // x - k = (x - round(x)) + (round(x) - k)
        nn0[h] = (float)(kr - k_lo);
        const float u0h = frx[h] + nn0[h];
        xf[h] = (float)tp.x;
        // phases in turns, reduced in fp64 (phi reaches ~1e8 rad), then to [-1/2, 1/2)
        double tphi = T.phic_turns - tp.X58 * (1.0 / kPi);
        tphi -= floor(tphi);
        double tpsi = 0.5 * tp.c + fr;
        tpsi -= floor(tpsi);
        float sphi, cphi, spsi, cpsi;
        __sincosf(6.283185307179586f * ((float)tphi - 0.5f), &sphi, &cphi);     // = -(sin, cos)(2 pi tphi)
        __sincosf(6.283185307179586f * ((float)tpsi - 0.5f), &spsi, &cpsi);
        const float cf = (float)tp.c;
        sc[h] = rsqrt_approx(0.5f * cf);
        kap[h] = 0.5f * cf * sc[h];                                             // sqrt(c/2)
        cc[h] = cf;
        hc[h] = 0.5f * rcp_approx(cf);
        const float pre = -(T.acoef * tp.Xm14) * (0.5f * sc[h]);              // -A_m / sqrt(2c)
        Pr[h] = pre * cphi;
        Pi[h] = pre * sphi;
        Er[h] = -cpsi;
        Ei[h] = -spsi;
        // near zone: offsets j with |v0| < kVFar or |v1| < kVFar, i.e. -(c + d) < u - j < d; FAR2 outside (j2a, j2b)
        const float d = fmaf(kVFar, kap[h], 1e-3f), d2 = fmaf(kVFar2, kap[h], 1e-3f);
        ja = min(ja, max(__float2int_rd(u0h - d) + 1, 0));
        jb = max(jb, __float2int_ru(u0h + cf + d));
        j2a = min(j2a, max(__float2int_rd(u0h - d2) + 1, 0));
        j2b = max(j2b, __float2int_ru(u0h + cf + d2));
      }
    }
    // transfer factors of the two channels (a6): constant per template, or from the template's table at f_m
    float vr[2] = {0.f, 0.f}, vi[2] = {0.f, 0.f}, vq[2] = {0.f, 0.f};
    if (__any_sync(0xffffffffu, any)) {
      const int Wmax = __reduce_max_sync(0xffffffffu, max(Wm[0], Wm[1]));
      const int Wmin = __reduce_min_sync(0xffffffffu, wmin);
      int JB = min(__reduce_max_sync(0xffffffffu, jb), Wmax);
      int JA = min(__reduce_min_sync(0xffffffffu, ja), JB);
      const int J2A = min(__reduce_min_sync(0xffffffffu, j2a), JA);
      const int J2B = max(min(__reduce_max_sync(0xffffffffu, j2b), Wmax), JB);
      if (CENSUS && lane == 0) {
        // measurement only: [0, Wmax) splits into FAR2 | FAR | NEAR | FAR | FAR2 at J2A <= JA <= JB <= J2B; 64 pixel slots per offset
        atomicAdd(a.census + 0, 64ull * (unsigned)(J2A + Wmax - J2B));
        atomicAdd(a.census + 1, 64ull * (unsigned)((JA - J2A) + (J2B - JB)));
        atomicAdd(a.census + 2, 64ull * (unsigned)(JB - JA));
      }

      // ---------------- pixel loop (a3-a5) ----------------
      PairTrack L;
      L.kap = pk(kap[0], kap[1]);
      L.kapf = pk(kap[0] * 0.318309886183790672f, kap[1] * 0.318309886183790672f);
      L.c = pk(cc[0], cc[1]);
      L.Er = pk(Er[0], Er[1]); L.Ei = pk(Ei[0], Ei[1]);
      L.sc = pk(sc[0], sc[1]); L.hc = pk(hc[0], hc[1]);
      SlabPair<WMODE> sl;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const unsigned col = (unsigned)(32 * h + lane);
        sl.y[h] = slab_y + ((unsigned)krel[h] * kTS + col) * 16u;
        sl.w[h] = WMODE == kWGeneral ? slab_w + ((unsigned)krel[h] * kTS + col) * 8u : slab_w + (unsigned)krel[h] * 8u;
#ifdef TFS_BOUNDS_CHECK
        sl.row_rel[h] = krel[h]; sl.rows = slab_rows(WMODE);
        if (krel[h] < 0 || krel[h] + Wmax > slab_rows(WMODE)) __trap();
#endif
      }
      PairSums s;
#pragma unroll
      for (int h = 0; h < 2; ++h) { s.zr[h] = pk(0.f, 0.f); s.zi[h] = pk(0.f, 0.f); s.q[h] = pk(0.f, 0.f); }
      const f2_t fr2 = pk(frx[0], frx[1]), n02 = pk(nn0[0], nn0[1]);
      const int Z2A = min(J2A, Wmin), ZA = min(JA, Wmin), ZB = min(JB, Wmin), Z2B = min(J2B, Wmin);
      // the zones may run in any order (u is re-derived from the offset), so the two FAR2 runs and the two
      // FAR runs share their code
#pragma unroll 1
      for (int r = 0; r < 2; ++r) pair_zone<kZFar2, WMODE>(sl, L, a.far, r ? Z2B : 0, r ? Wmin : Z2A, fr2, n02, lut_lane, s);
#pragma unroll 1
      for (int r = 0; r < 2; ++r) pair_zone<kZFar, WMODE>(sl, L, a.far, r ? ZB : Z2A, r ? Z2B : ZA, fr2, n02, lut_lane, s);
      pair_zone<kZNear, WMODE>(sl, L, a.far, ZA, ZB, fr2, n02, lut_lane, s);
      {
        // masked tail: a tranche whose window has ended contributes zero
        const float fw = (float)Wmin;
        f2_t nn = fadd2(n02, pk(-fw, -fw));
#pragma unroll 1
        for (int j = Wmin; j < Wmax; ++j) {
          const f2_t u = fadd2(fr2, nn);
          if (j >= JA && j < JB) pair_pixel<kZNear, WMODE, 1>(sl, L, a.far, j, u, Wm[0], Wm[1], lut_lane, s);
          else if (j < J2A || j >= J2B) pair_pixel<kZFar2, WMODE, 1>(sl, L, a.far, j, u, Wm[0], Wm[1], lut_lane, s);
          else pair_pixel<kZFar, WMODE, 1>(sl, L, a.far, j, u, Wm[0], Wm[1], lut_lane, s);
          nn = fadd2(nn, pk(-1.f, -1.f));
        }
      }
      // ---------------- a6: transfer factors, the tranche's factor P, weights a[i] ----------------
      float q0[2], q1[2];
      if (WMODE == kWTimeOnly) {
        float r0, r1, s0, s1;
        upk(s.q[0], r0, r1); upk(s.q[1], s0, s1);              // {sum hr^2, sum hi^2} per half
        q0[0] = q1[0] = r0 + s0;
        q0[1] = q1[1] = r1 + s1;
      } else {
        upk(s.q[0], q0[0], q1[0]);
        upk(s.q[1], q0[1], q1[1]);
      }
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        float T0r = T.T0r, T0i = T.T0i, T1r = T.T1r, T1i = T.T1i;
        if (a.ttab != nullptr) {
          // T_alpha(f_m) from the template's table: linear between knots, clamped outside (Eq. 29)
          const int K = a.tt_K;
          float sx = fmaf(xf[h], a.tt_scale, -a.tt_off);
          sx = fminf(fmaxf(sx, 0.f), (float)(K - 1));
          const int kn = min((int)sx, max(K - 2, 0));
          const float tf = K > 1 ? sx - (float)kn : 0.f;
          const int kn1 = min(kn + 1, K - 1);
          const float2* tb = a.ttab + ((size_t)it * a.tt_C + a.tt_ch0) * K;
          const float2 A0 = __ldg(tb + kn), A1 = __ldg(tb + kn1);
          T0r = fmaf(tf, A1.x - A0.x, A0.x); T0i = fmaf(tf, A1.y - A0.y, A0.y);
          T1r = 0.f; T1i = 0.f;
          if (a.tt_ch0 + 1 < a.tt_C && a.n_ch_pair > 1) {
            const float2 B0 = __ldg(tb + K + kn), B1 = __ldg(tb + K + kn1);
            T1r = fmaf(tf, B1.x - B0.x, B0.x); T1i = fmaf(tf, B1.y - B0.y, B0.y);
          }
        }
        // z' = T_0 z'_0 + T_1 z'_1 ;  q' = |T_0|^2 a_0 q'_0 + |T_1|^2 a_1 q'_1   (Eq. 29, Eq. 31)
        const f2_t Tr = pk(T0r, T1r), Ti = pk(T0i, T1i);
        float ar, br, ai, bi;
        upk(ffma2(Ti ^ 0x8000000080000000ULL, s.zi[h], fmul2(Tr, s.zr[h])), ar, br);     // T.re z.re - T.im z.im per channel
        upk(ffma2(Ti, s.zr[h], fmul2(Tr, s.zi[h])), ai, bi);                             // T.re z.im + T.im z.re
        const float zcr = ar + br, zci = ai + bi;
        f2_t w2 = ffma2(Tr, Tr, fmul2(Ti, Ti));                                           // |T|^2 per channel
        if (WMODE != kWGeneral) {
          const float2 am = __ldg(a.wa + idxv[h]);
          w2 = fmul2(w2, pk(am.x, am.y));
        }
        float w0, w1;
        upk(w2, w0, w1);
        const float P2 = fmaf(Pr[h], Pr[h], Pi[h] * Pi[h]);
        vr[h] = fmaf(Pr[h], zcr, -Pi[h] * zci);                  // Re (P z')
        vi[h] = fmaf(Pr[h], zci, Pi[h] * zcr);                   // Im (P z')
        vq[h] = P2 * fmaf(w0, q0[h], w1 * q1[h]);
      }
    }

    // ---------------- a7: pieces.  Chunk h covers entries [i0 + 32 h, ...): add its lanes to the current piece;
    // every piece that ends inside the chunk (a segment boundary, or the end of the tile) takes the lanes
    // before its end and is closed; the lanes behind the last such end open the next piece ----------------
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int ic = i0 + 32 * h;
      if (ic >= i1) break;
      const int cend = min(ic + 32, i1);
      if (!(p < p_stop && pend <= cend)) { accr += vr[h]; acci += vi[h]; acch += vq[h]; continue; }
      int lo = 0;
      for (;;) {
        const bool ends = p < p_stop && pend <= cend;
        const int hi = ends ? pend - ic : 32;
        if (lane >= lo && lane < hi) { accr += vr[h]; acci += vi[h]; acch += vq[h]; }
        if (!ends) break;
        // close piece p: sum the lanes (fp32 butterfly: 32 terms), store, reset
        float r0 = accr, r1 = acci, r2 = acch;
        accr = 0.f; acci = 0.f; acch = 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          r0 += __shfl_xor_sync(0xffffffffu, r0, o);
          r1 += __shfl_xor_sync(0xffffffffu, r1, o);
          r2 += __shfl_xor_sync(0xffffffffu, r2, o);
        }
        if (lane == 0) {
          float4* dst = a.partials + (long long)p * a.n + it;
          float4 v = make_float4(r0, r1, r2, 0.f);
          if (a.accumulate) { const float4 o = *dst; v.x += o.x; v.y += o.y; v.z += o.z; }
          *dst = v;
        }
        ++p;
        if (p < p_stop) pend = a.piece_end[p];
        lo = hi;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// mbarrier / TMA primitives (PTX ISA: mbarrier, cp.async.bulk, cp.async.bulk.tensor)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_2d(unsigned dst, const CUtensorMap* map, int c0, int c1, unsigned bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
               :: "r"(dst), "l"((unsigned long long)map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_load_1d(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(dst), "l"((unsigned long long)src), "r"(bytes), "r"(bar) : "memory");
}

// dynamic shared memory of the slab kernel
//   [LUT: (kLutN+1) * kLutCopiesSlab float4][stage 0][stage 1][control]
//   stage = data slab [rows][kTS] float4, then (kWGeneral) weight slab [rows][kTS] float2
//           or (kWSeparable) rows of the b table [rows] float2
constexpr int kLutSlabBytes = ((kLutN + 1) * kLutCopiesSlab * (int)sizeof(float4) + 127) / 128 * 128;   // slabs start 128-byte aligned
__host__ __device__ constexpr int slab_y_bytes(int wmode) { return slab_rows(wmode) * kTS * 16; }
__host__ __device__ constexpr int slab_w_bytes(int wmode) {
  return wmode == kWGeneral ? slab_rows(wmode) * kTS * 8 : (wmode == kWSeparable ? slab_rows(wmode) * 8 : 0);
}
__host__ __device__ constexpr int slab_stage_bytes(int wmode) { return (slab_y_bytes(wmode) + slab_w_bytes(wmode) + 127) / 128 * 128; }
constexpr int kSlabCtlBytes = 128;        // full[2], empty[2] mbarriers, 2 unit descriptors, 2 item counters
__host__ __device__ constexpr int slab_smem_bytes(int wmode) { return kLutSlabBytes + 2 * slab_stage_bytes(wmode) + kSlabCtlBytes; }
static_assert(slab_smem_bytes(kWGeneral) <= 232448 && slab_smem_bytes(kWSeparable) <= 232448, "slab kernel exceeds 227 KB of shared memory");

struct SlabCtl {
  unsigned long long full[2], empty[2];
  Unit unit[2];
  unsigned next_item[2];
};
static_assert(sizeof(SlabCtl) <= kSlabCtlBytes, "SlabCtl");

// ------------------------------------------------------------------------------------------
// eval_slab_kernel: persistent, one CTA of 32 warps per SM.  Thread 0 is also the producer: it claims the
// next unit from the global counter, posts its descriptor and issues the TMA copies of the band's slab
// into the stage's buffer; the stage's `full` mbarrier completes when the bytes have landed.  Every warp
// then takes items of the unit from the stage's counter until it is exhausted, arrives on the stage's
// `empty` mbarrier and moves on to the other stage; the producer refills a stage once all 32 warps have
// left it.  Units come in tile-major, band-major order, so consecutive units mostly reload the same slab
// from the L2.
// ------------------------------------------------------------------------------------------
template <int WMODE, bool CENSUS = false>      // CENSUS: the measurement build of tfs_tier_census (the default build carries no counting code)
__global__ void __launch_bounds__(kSlabWarps * 32, 1)
eval_slab_kernel(const EvalArgs a, const __grid_constant__ CUtensorMap map_y, const __grid_constant__ CUtensorMap map_w) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float4* s_lut = reinterpret_cast<float4*>(smem_raw);
  SlabCtl* ctl = reinterpret_cast<SlabCtl*>(smem_raw + kLutSlabBytes + 2 * slab_stage_bytes(WMODE));
  const unsigned smem_base = (unsigned)__cvta_generic_to_shared(smem_raw);
  const unsigned stage_base = smem_base + kLutSlabBytes;
  const unsigned ctl_base = stage_base + 2 * slab_stage_bytes(WMODE);
  const unsigned bar_full = ctl_base + (unsigned)offsetof(SlabCtl, full);
  const unsigned bar_empty = ctl_base + (unsigned)offsetof(SlabCtl, empty);
  constexpr int R = slab_rows(WMODE);

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < (kLutN + 1) * kLutCopiesSlab; i += blockDim.x) s_lut[i] = a.lut[i / kLutCopiesSlab];
  if (threadIdx.x == 0) {
    mbar_init(bar_full, 1); mbar_init(bar_full + 8, 1);
    mbar_init(bar_empty, kSlabWarps); mbar_init(bar_empty + 8, kSlabWarps);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const unsigned lut_lane = smem_base + 16u * (unsigned)(lane & (kLutCopiesSlab - 1)) - kMagicBits * (16u * kLutCopiesSlab);
  const int n_units = a.n_units[0];

  // producer: claim the next unit and fill stage s with it
  auto produce = [&](int s) {
    const unsigned long long uid = atomicAdd(a.work_counter, 1ULL);
    Unit d;
    if (uid < (unsigned long long)n_units) d = a.units_slab[uid];
    else { d.tile = 0; d.row0 = 0; d.off = 0; d.cnt = -1; }
    ctl->unit[s] = d;
    ctl->next_item[s] = 0;
    const unsigned bar = bar_full + 8u * s;
    if (d.cnt < 0) { mbar_arrive(bar); return; }
    const unsigned dst = stage_base + (unsigned)s * slab_stage_bytes(WMODE);
    mbar_arrive_expect_tx(bar, (unsigned)(slab_y_bytes(WMODE) + slab_w_bytes(WMODE)));
    tma_load_2d(dst, &map_y, d.tile * kTS * 4, d.row0, bar);
    if (WMODE == kWGeneral) tma_load_2d(dst + slab_y_bytes(WMODE), &map_w, d.tile * kTS * 2, d.row0, bar);
    if (WMODE == kWSeparable) bulk_load_1d(dst + slab_y_bytes(WMODE), a.wb + d.row0, R * 8, bar);
  };
  if (threadIdx.x == 0) { produce(0); produce(1); }

  int stage = 0;
  unsigned phase = 0;
  for (;;) {
    mbar_wait(bar_full + 8u * stage, phase);
    const Unit d = ctl->unit[stage];
    if (d.cnt < 0) break;
    const unsigned slab_y = stage_base + (unsigned)stage * slab_stage_bytes(WMODE);
    const unsigned slab_w = slab_y + slab_y_bytes(WMODE);
    for (;;) {
      int k = 0;
      if (lane == 0) k = (int)atomicAdd(&ctl->next_item[stage], 1u);
      k = __shfl_sync(0xffffffffu, k, 0);
      if (k >= d.cnt) break;
      const long long it = (long long)a.list[d.off + (unsigned)k];
      eval_item_pair<WMODE, CENSUS>(a, it, d.tile, lane, lut_lane, slab_y, slab_w, d.row0);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_empty + 8u * stage);
    if (warp == 0) {
      if (lane == 0) {
        mbar_wait(bar_empty + 8u * stage, phase);       // all 32 warps have left the stage
        produce(stage);
      }
      __syncwarp();
    }
    stage ^= 1;
    if (stage == 0) phase ^= 1u;
  }
}

// ------------------------------------------------------------------------------------------
// eval_list_kernel: the items the slab kernel cannot take (and every item when fresnel_mode = 1).
// Persistent: one CTA per SM, warps claim units of <= kListUnitItems items of one tile, in tile-major
// order so that the tile's columns stay L2-resident, and gather from global memory.
// ------------------------------------------------------------------------------------------
constexpr int kLutListBytes = (kLutN + 1) * kLutCopiesList * (int)sizeof(float4);

template <int MODE, int WMODE, bool CENSUS = false>
__global__ void __launch_bounds__(kWarpsPerCta * 32, 1)
eval_list_kernel(const EvalArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float4* s_lut = reinterpret_cast<float4*>(smem_raw);
  const int lane = threadIdx.x & 31;
  if (MODE != 1) {
    for (int i = threadIdx.x; i < (kLutN + 1) * kLutCopiesList; i += blockDim.x) s_lut[i] = a.lut[i / kLutCopiesList];
    __syncthreads();
  }
  const unsigned lut_lane = (unsigned)__cvta_generic_to_shared(s_lut) + 16u * (unsigned)(lane & (kLutCopiesList - 1)) -
                            kMagicBits * (16u * kLutCopiesList);
  const int n_units = a.n_units[1];
  for (;;) {
    unsigned long long uid = 0;
    if (lane == 0) uid = atomicAdd(a.work_counter + 1, 1ULL);
    uid = __shfl_sync(0xffffffffu, uid, 0);
    if (uid >= (unsigned long long)n_units) break;
    const Unit d = a.units_list[uid];
    for (int k = 0; k < d.cnt; ++k) {
      const long long it = (long long)a.list[d.off + (unsigned)k];
      eval_item<MODE, WMODE, CENSUS>(a, it, d.tile, lane, lut_lane);
    }
  }
}

// ------------------------------------------------------------------------------------------
// Pre-pass (per batch).
// ------------------------------------------------------------------------------------------
__global__ void prep_consts_kernel(const EvalArgs a) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.n) return;
  TplConst t = load_template(a.params + i * 8, a.DT, a.t_col, a.n_ch_pair);
  if (a.t_col < 0 && t.ok) { t.T0r = (float)a.t3_re; t.T0i = (float)a.t3_im; }
  a.tconst[i] = t;
  if (a.bad_count != nullptr && !t.ok) atomicAdd(a.bad_count, 1ULL);
}

// Bucket of item (template i, tile t), from the track at the tile's first and last valid tranche (x and c
// grow with time, so they bound every tranche in between):
//   0  no tranche of the tile can be active (merged before the tile, above the band or too fast at its
//      start, below the band at its end, bad row): the item is skipped and its partials are never read;
//   1  list kernel: the template merges inside the tile, or the rows its lanes can touch
//      [k_lo(first), ceil(x_last) + floor(c_last) + H + 3] do not fit the slab of its band (a lane reads
//      Wmax <= floor(c_last) + 2H + 2 rows from its own k_lo <= ceil(x_last) - H, the longest window of its
//      chunk; rows past Nf + kPadRows do not exist and the TMA copy fills them with zeros);
//   2+b  slab kernel, band b = k_lo(first) / kBandStride.
// The skip tests carry a relative slack of 1e-9, so an item is never dropped on a rounding difference
// against the per-lane tests (an item kept needlessly just yields zeros).
__device__ __forceinline__ int item_key(const EvalArgs& a, const TplConst& T, int tile) {
  if (!T.ok) return 0;
  const int i0 = tile * kTS, i1 = min(i0 + kTS, a.n_valid);
  if (i0 >= i1) return 0;
  const int m0 = a.valid_m[i0], m1 = a.valid_m[i1 - 1];
  if (a.basis == 1) {
    // WDM pixels (tfs_wdm.cuh): the same monotone bounds with the WDM activity rule; always the list path
    const double sl = 1.0 + 1e-9;
    const TrackPoint w0 = track_point_at(T, (double)m0 * a.wdm_DTpix, a.DT, -1.0, 1e300, 1e300, 0.0, true);
    if (!w0.active) return 0;
    if (w0.x + 0.5 * w0.c > a.x_hi * sl || w0.c > a.c_max * sl) return 0;
    const TrackPoint w1 = track_point_at(T, (double)m1 * a.wdm_DTpix, a.DT, -1.0, 1e300, 1e300, 0.0, true);
    if (w1.active && w1.x * sl < a.x_lo) return 0;
    return 1;
  }
  const TrackPoint t0 = track_point(T, m0, a.DT, -1.0, 1e300, 1e300, true);
  if (!t0.active) return 0;                                        // tau <= DT at the tile's start
  const double slack = 1.0 + 1e-9;
  if (t0.x + t0.c > a.x_hi * slack || t0.c > a.c_max * slack) return 0;
  const TrackPoint t1 = track_point(T, m1, a.DT, -1.0, 1e300, 1e300, true);
  if (!t1.active) return 1;                                        // merges inside the tile
  if (t1.x * slack < a.x_lo) return 0;
  if (!a.slab_ok) return 1;
  if (!(t1.c <= 1e6) || !(t1.x <= 2.0e9)) return 1;
  const int klo = min(max((int)ceil(t0.x) - a.H, 1), a.Nf - 1);
  int ktop = (int)ceil(t1.x) + (a.adaptive ? (int)floor(t1.c) : 0) + a.H + 3;
  const int b = klo / kBandStride;
  if (ktop >= b * kBandStride + slab_rows(a.wmode) || ktop < klo) return 1;
  return 2 + b;
}

// grid (ceil(n/(256 kPrepItems)), n_tiles): keys of the tile's items + the tile's bucket counts; every thread takes
// kPrepItems templates (strided by the block size: coalesced) so that the per-block histogram work -- zeroing and
// flushing n_keys (~200) shared counters -- is paid once per 1024 items
constexpr int kPrepItems = 4;
__global__ void __launch_bounds__(256)
prep_keys_kernel(const EvalArgs a) {
  extern __shared__ unsigned s_hist[];                              // [n_keys]
  for (int k = threadIdx.x; k < a.n_keys; k += blockDim.x) s_hist[k] = 0;
  __syncthreads();
  const int tile = blockIdx.y;
#pragma unroll 1
  for (int q = 0; q < kPrepItems; ++q) {
    const long long i = ((long long)blockIdx.x * kPrepItems + q) * blockDim.x + threadIdx.x;
    if (i < a.n) {
      const int key = item_key(a, a.tconst[i], tile);
      a.keys[(size_t)tile * a.n + i] = (uint16_t)key;
      if (key) atomicAdd(&s_hist[key], 1u);
    }
  }
  __syncthreads();
  for (int k = threadIdx.x; k < a.n_keys; k += blockDim.x)
    if (s_hist[k]) atomicAdd(&a.counts[(size_t)tile * a.n_keys + k], s_hist[k]);
}

// one CTA: exclusive scan of the bucket counts (tile-major, key-major) -> bucket_off; unit tables; the
// counts are zeroed (they become the scatter cursors)
__global__ void __launch_bounds__(1024)
prep_scan_kernel(const EvalArgs a) {
  __shared__ unsigned s_items[1024], s_us[1024], s_ul[1024];
  const int nb = a.n_tiles * a.n_keys;
  const int per = (nb + 1023) / 1024;
  const int b0 = min((int)threadIdx.x * per, nb), b1 = min(b0 + per, nb);
  unsigned items = 0, us = 0, ul = 0;
  for (int b = b0; b < b1; ++b) {
    const int key = b % a.n_keys;
    const unsigned c = key ? a.counts[b] : 0u;
    items += c;
    if (key >= 2) us += (c + kUnitItems - 1) / kUnitItems;
    if (key == 1) ul += (c + kListUnitItems - 1) / kListUnitItems;
  }
  s_items[threadIdx.x] = items; s_us[threadIdx.x] = us; s_ul[threadIdx.x] = ul;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {                             // inclusive Hillis-Steele scans
    unsigned v0 = 0, v1 = 0, v2 = 0;
    if ((int)threadIdx.x >= o) { v0 = s_items[threadIdx.x - o]; v1 = s_us[threadIdx.x - o]; v2 = s_ul[threadIdx.x - o]; }
    __syncthreads();
    s_items[threadIdx.x] += v0; s_us[threadIdx.x] += v1; s_ul[threadIdx.x] += v2;
    __syncthreads();
  }
  unsigned off = s_items[threadIdx.x] - items, iu = s_us[threadIdx.x] - us, il = s_ul[threadIdx.x] - ul;
  for (int b = b0; b < b1; ++b) {
    const int key = b % a.n_keys, tile = b / a.n_keys;
    const unsigned c = key ? a.counts[b] : 0u;
    a.bucket_off[b] = off;
    a.counts[b] = 0;
    if (key >= 2) {
      for (unsigned o = 0; o < c; o += kUnitItems) {
        Unit u; u.tile = tile; u.row0 = (key - 2) * kBandStride; u.off = off + o; u.cnt = (int)min(c - o, (unsigned)kUnitItems);
        a.units_slab[iu++] = u;
      }
    } else if (key == 1) {
      for (unsigned o = 0; o < c; o += kListUnitItems) {
        Unit u; u.tile = tile; u.row0 = 0; u.off = off + o; u.cnt = (int)min(c - o, (unsigned)kListUnitItems);
        a.units_list[il++] = u;
      }
    }
    off += c;
  }
  if (threadIdx.x == 1023) { a.n_units[0] = (int)s_us[1023]; a.n_units[1] = (int)s_ul[1023]; }
}

// grid as prep_keys_kernel: template indices into their bucket's range of `list` (order inside a bucket is
// arbitrary: every item writes its own partials, so the results do not depend on it)
__global__ void __launch_bounds__(256)
prep_scatter_kernel(const EvalArgs a) {
  extern __shared__ unsigned s_hist[];                              // [2][n_keys]: count, then base
  unsigned* s_cnt = s_hist;
  unsigned* s_base = s_hist + a.n_keys;
  for (int k = threadIdx.x; k < a.n_keys; k += blockDim.x) s_cnt[k] = 0;
  __syncthreads();
  const int tile = blockIdx.y;
  int key[kPrepItems];
  unsigned rank[kPrepItems];
#pragma unroll
  for (int q = 0; q < kPrepItems; ++q) {
    const long long i = ((long long)blockIdx.x * kPrepItems + q) * blockDim.x + threadIdx.x;
    key[q] = 0; rank[q] = 0;
    if (i < a.n) {
      key[q] = a.keys[(size_t)tile * a.n + i];
      if (key[q]) rank[q] = atomicAdd(&s_cnt[key[q]], 1u);
    }
  }
  __syncthreads();
  for (int k = threadIdx.x; k < a.n_keys; k += blockDim.x)
    if (s_cnt[k]) s_base[k] = atomicAdd(&a.counts[(size_t)tile * a.n_keys + k], s_cnt[k]);
  __syncthreads();
#pragma unroll
  for (int q = 0; q < kPrepItems; ++q) {
    const long long i = ((long long)blockIdx.x * kPrepItems + q) * blockDim.x + threadIdx.x;
    if (key[q]) a.list[a.bucket_off[(size_t)tile * a.n_keys + key[q]] + s_base[key[q]] + rank[q]] = (unsigned)i;
  }
}

// Piece table (C9, C10).  Segment n = tranches [ceil(n Nt/N_seg), ceil((n+1) Nt/N_seg)), i.e. n(m) =
// floor(m N_seg / Nt); or, with M_tr > 0 (tfs_eval_tseg: segments of fixed duration T_seg = M_tr DT, t_n = n T_seg,
// P:93), n(m) = floor(m / M_tr) and N_seg = ceil(Nt / M_tr).  Tile t = entries [t kTS, (t+1) kTS) of the compacted valid-tranche list.
// A piece is a maximal run of entries inside one tile and one segment; pieces are numbered in time order.
// One thread walks the list (<= n_tiles + N_seg pieces); the table is cached per N_seg by the host.
//   tile_first[t] = first piece of tile t, tile_first[n_tiles] = number of pieces
//   piece_end[p]  = entry where piece p ends (exclusive);  piece_seg[p] = its segment;  piece_tile[p] = its tile
__global__ void piece_table_kernel(const int* __restrict__ vprefix, const int* __restrict__ valid_m, int Nt, int N_seg,
                                   int M_tr, int n_valid, int n_tiles, int* __restrict__ tile_first,
                                   int* __restrict__ piece_end, int* __restrict__ piece_seg, int* __restrict__ piece_tile) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  int p = 0;
  for (int t = 0; t < n_tiles; ++t) {
    tile_first[t] = p;
    int i = t * kTS;
    const int iend = min(i + kTS, n_valid);
    while (i < iend) {
      const int seg = M_tr > 0 ? valid_m[i] / M_tr : (int)(((long long)valid_m[i] * N_seg) / Nt);
      const long long s1l = M_tr > 0 ? (long long)(seg + 1) * M_tr
                                     : ((long long)(seg + 1) * Nt + N_seg - 1) / N_seg;   // first tranche of the next segment
      const int s1 = (int)(s1l < (long long)Nt ? s1l : (long long)Nt);
      const int e = min(vprefix[min(s1, Nt)], iend);
      piece_seg[p] = seg;
      piece_end[p] = e;
      piece_tile[p] = t;
      ++p;
      i = e;
    }
  }
  tile_first[n_tiles] = p;
}

// ------------------------------------------------------------------------------------------
// combine_kernel: sum the piece partials of each segment, P_n = |z_n|^2/hh_n, Upsilon = sum_n P_n
// (Eq. 8, 9), fp64.  Pieces are in time order, so the pieces of a segment are consecutive; a segment
// without a valid tranche has no piece and contributes 0; the partials of an item whose bucket is 0 were
// never written and are not read.
// ------------------------------------------------------------------------------------------
__global__ void combine_kernel(const float4* __restrict__ partials, const uint16_t* __restrict__ keys, long long n, int N_seg,
                               const int* __restrict__ tile_first, int n_tiles, const int* __restrict__ piece_seg,
                               const int* __restrict__ piece_tile,
                               float* __restrict__ upsilon, float* __restrict__ seg_power,
                               float* __restrict__ seg_dh, float* __restrict__ seg_hh, int* __restrict__ n_seg_eff) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int n_pieces = tile_first[n_tiles];
  double ups = 0.0;
  int p = 0, cur_tile = -1, n_eff = 0;
  bool live = false;
  for (int s = 0; s < N_seg; ++s) {
    double zr = 0, zi = 0, hh = 0;
    for (; p < n_pieces && piece_seg[p] == s; ++p) {
      const int t = piece_tile[p];
      if (t != cur_tile) { cur_tile = t; live = keys[(size_t)t * n + i] != 0; }
      if (!live) continue;
      const float4 v = partials[(long long)p * n + i];
      zr += v.x; zi += v.y; hh += v.z;
    }
    const double P = hh > 0.0 ? (zr * zr + zi * zi) / hh : 0.0;
    ups += P;
    n_eff += hh > 0.0 ? 1 : 0;
    if (seg_power) seg_power[i * N_seg + s] = (float)P;
    if (seg_dh) { seg_dh[(i * N_seg + s) * 2] = (float)zr; seg_dh[(i * N_seg + s) * 2 + 1] = (float)zi; }
    if (seg_hh) seg_hh[i * N_seg + s] = (float)hh;
  }
  upsilon[i] = (float)ups;
  if (n_seg_eff) n_seg_eff[i] = n_eff;      // segments the template occupies: the paper's N_seg = tau / T_seg
}

// ------------------------------------------------------------------------------------------
// Window pixel counts (phase 1 only).
// ------------------------------------------------------------------------------------------
__global__ void count_pixels_kernel(const EvalArgs a, long long* __restrict__ counts) {
  const int lane = threadIdx.x & 31;
  const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= a.n) return;
  const TplConst T = load_template(a.params + w * 8, a.DT, -1, 0);
  long long cnt = 0;
  if (T.ok) {
    for (int m = lane; m < a.Nt; m += 32) {
      const TrackPoint tp = track_point(T, m, a.DT, a.x_lo, a.x_hi, a.c_max, a.gap[m] != 0);
      if (tp.active) {
        int k_lo, k_hi;
        window(tp, a.H, a.adaptive, a.Nf, k_lo, k_hi);
        cnt += k_hi - k_lo + 1;
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  if (lane == 0) counts[w] = cnt;
}

// ------------------------------------------------------------------------------------------
// Upload (a0): Y = W*D interleaved by channel and W interleaved, transposed to time-contiguous [k][i]
// over the compacted list of valid tranches (i = vprefix[m]; gap tranches are not stored) through a
// 32x32 shared-memory tile (reads coalesced along k, writes coalesced along i).  Channel c1 < 0: the
// second half of the pair is empty (zeros).  The arrays are zeroed before this kernel runs, so pad rows
// and pad columns stay zero.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
pack_kernel(const float2* __restrict__ coeff, const float* __restrict__ weight, const float* __restrict__ bk, int Nt, int Nf,
            int c0, int c1, const uint8_t* __restrict__ gap, const int* __restrict__ vprefix, int ncol,
            float4* __restrict__ grid, float2* __restrict__ wgt) {
  __shared__ float4 sY[32][33];
  __shared__ float2 sW[32][33];
  const int k0 = blockIdx.x * 32, m0 = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;        // 32 x 8
  const long long npix = (long long)Nt * Nf;
  for (int r = ty; r < 32; r += 8) {
    const int m = m0 + r, k = k0 + tx;
    if (m < Nt && k < Nf) {
      const long long i = (long long)m * Nf + k;
      float2 dA = coeff[c0 * npix + i], dE = c1 >= 0 ? coeff[c1 * npix + i] : make_float2(0.f, 0.f);
      // W: the per-pixel array; or (front end, weights known to be W[a,m,k] = bk[a][k]) the per-bin table; or 1
      float wA = weight ? weight[c0 * npix + i] : (bk ? bk[(size_t)c0 * Nf + k] : 1.0f);
      float wE = c1 >= 0 ? (weight ? weight[c1 * npix + i] : (bk ? bk[(size_t)c1 * Nf + k] : 1.0f)) : 0.f;
      // a pixel whose product W*D is not finite carries no information: weight 0 (also keeps every
      // value the gather can read finite, which the pixel loops rely on)
      if (!(isfinite(wA * dA.x) && isfinite(wA * dA.y) && isfinite(wA))) { wA = 0.f; dA = make_float2(0.f, 0.f); }
      if (!(isfinite(wE * dE.x) && isfinite(wE * dE.y) && isfinite(wE))) { wE = 0.f; dE = make_float2(0.f, 0.f); }
      sY[r][tx] = make_float4(wA * dA.x, wE * dE.x, wA * dA.y, wE * dE.y);
      sW[r][tx] = make_float2(wA, wE);
    }
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const int k = k0 + r, m = m0 + tx;
    if (m < Nt && k < Nf && gap[m] != 0) {
      const long long o = (long long)k * ncol + vprefix[m];
      grid[o] = sY[tx][r];
      if (wgt) wgt[o] = sW[tx][r];
    }
  }
}

// ------------------------------------------------------------------------------------------
// Weight structure (a0, C11), over the valid tranches.  If W[alpha,i,k] = a_alpha[i] b_alpha[k] then
//   rowmax[i] = max_k W = a[i] max b,  colmax[k] = max_i W = b[k] max a,  gmax = max a max b,
// so a'[i] = rowmax[i], b'[k] = colmax[k] / gmax reproduce W = a' b'.  weight_check_kernel counts the
// pixels where that fails by more than a few ulps (or W < 0), and the columns with b' != 1.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
weight_colmax_kernel(const float2* __restrict__ wgt, int ncol, int n_valid, float2* __restrict__ colmax) {   // one block per k
  __shared__ float2 sh[256];
  const int k = blockIdx.x;
  float2 mx = make_float2(0.f, 0.f);
  for (int m = threadIdx.x; m < n_valid; m += 256) {
    const float2 w = wgt[(size_t)k * ncol + m];
    mx.x = fmaxf(mx.x, w.x); mx.y = fmaxf(mx.y, w.y);
  }
  sh[threadIdx.x] = mx;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sh[threadIdx.x].x = fmaxf(sh[threadIdx.x].x, sh[threadIdx.x + o].x);
      sh[threadIdx.x].y = fmaxf(sh[threadIdx.x].y, sh[threadIdx.x + o].y);
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) colmax[k] = sh[0];
}

// wa must be zeroed first; grid (ceil(n_valid/128), k-slices): weights are >= 0 (or zeroed at upload), so their
// bit patterns order like integers and atomicMax on them is the float maximum
__global__ void weight_rowmax_kernel(const float2* __restrict__ wgt, int ncol, int n_valid, int Nf, float2* __restrict__ wa) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n_valid) return;
  const int per = (Nf + gridDim.y - 1) / gridDim.y;
  const int k0 = blockIdx.y * per, k1 = min(k0 + per, Nf);
  float2 mx = make_float2(0.f, 0.f);
  for (int k = k0; k < k1; ++k) {
    const float2 w = wgt[(size_t)k * ncol + m];
    mx.x = fmaxf(mx.x, w.x); mx.y = fmaxf(mx.y, w.y);
  }
  int* out = reinterpret_cast<int*>(wa + m);
  atomicMax(out, __float_as_int(fmaxf(mx.x, 0.f)));
  atomicMax(out + 1, __float_as_int(fmaxf(mx.y, 0.f)));
}

// one block: gmax = max_k colmax[k]; wb[k] = colmax[k] / gmax (0 where gmax = 0); counts[1] += #{b' != 1}
__global__ void __launch_bounds__(1024)
weight_factor_kernel(const float2* __restrict__ colmax, int Nf, float2* __restrict__ wb, unsigned long long* counts) {
  __shared__ float2 sh[1024];
  float2 mx = make_float2(0.f, 0.f);
  for (int k = threadIdx.x; k < Nf; k += 1024) { mx.x = fmaxf(mx.x, colmax[k].x); mx.y = fmaxf(mx.y, colmax[k].y); }
  sh[threadIdx.x] = mx;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sh[threadIdx.x].x = fmaxf(sh[threadIdx.x].x, sh[threadIdx.x + o].x);
      sh[threadIdx.x].y = fmaxf(sh[threadIdx.x].y, sh[threadIdx.x + o].y);
    }
    __syncthreads();
  }
  const float2 g = sh[0];
  unsigned long long not_one = 0;
  for (int k = threadIdx.x; k < Nf; k += 1024) {
    const float2 b = make_float2(g.x > 0.f ? colmax[k].x / g.x : 0.f, g.y > 0.f ? colmax[k].y / g.y : 0.f);
    wb[k] = b;
    not_one += (g.x > 0.f && b.x != 1.0f) + (g.y > 0.f && b.y != 1.0f);
  }
  if (not_one) atomicAdd(&counts[1], not_one);
}

__global__ void weight_check_kernel(const float2* __restrict__ wgt, const float2* __restrict__ wa,
                                    const float2* __restrict__ wb, int ncol, int n_valid, int Nf, unsigned long long* counts) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = false;
  if (i < (size_t)ncol * Nf) {
    const int k = (int)(i / ncol), m = (int)(i - (size_t)k * ncol);
    if (m < n_valid) {
      const float2 w = wgt[i], a = wa[m], b = wb[k];
      const float pA = a.x * b.x, pE = a.y * b.y;
      bad = !(fabsf(w.x - pA) <= 1e-6f * pA) || !(fabsf(w.y - pE) <= 1e-6f * pE) || w.x < 0.f || w.y < 0.f;
    }
  }
  const unsigned n_bad = __popc(__ballot_sync(0xffffffffu, bad));
  if ((threadIdx.x & 31) == 0 && n_bad) atomicAdd(&counts[0], (unsigned long long)n_bad);
}

// Separable weights known by construction (tfs_upload_timeseries: W[a,m,k] = bk[a][k], one PSD model per channel,
// or 1 without a PSD): fill a[i] = g = max_k bk, b[k] = bk[k]/g directly -- no per-pixel weight array is written,
// read or analysed.  One CTA.  counts[1] = number of bins with b != 1 (-> kWSeparable, else kWTimeOnly).
__global__ void __launch_bounds__(1024)
weight_sep_set_kernel(const float* __restrict__ bk, int Nf, int c0, int c1, int n_valid, float2* __restrict__ wa,
                      float2* __restrict__ wb, unsigned long long* counts) {
  __shared__ float2 sh[1024];
  float2 mx = make_float2(0.f, 0.f);
  for (int k = threadIdx.x; k < Nf; k += 1024) {
    const float bA = bk ? bk[(size_t)c0 * Nf + k] : 1.0f, bE = c1 >= 0 ? (bk ? bk[(size_t)c1 * Nf + k] : 1.0f) : 0.f;
    mx.x = fmaxf(mx.x, isfinite(bA) ? bA : 0.f); mx.y = fmaxf(mx.y, isfinite(bE) ? bE : 0.f);
  }
  sh[threadIdx.x] = mx;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sh[threadIdx.x].x = fmaxf(sh[threadIdx.x].x, sh[threadIdx.x + o].x);
      sh[threadIdx.x].y = fmaxf(sh[threadIdx.x].y, sh[threadIdx.x + o].y);
    }
    __syncthreads();
  }
  const float2 g = sh[0];
  unsigned long long not_one = 0;
  for (int k = threadIdx.x; k < Nf; k += 1024) {
    float bA = bk ? bk[(size_t)c0 * Nf + k] : 1.0f, bE = c1 >= 0 ? (bk ? bk[(size_t)c1 * Nf + k] : 1.0f) : 0.f;
    if (!isfinite(bA)) bA = 0.f;
    if (!isfinite(bE)) bE = 0.f;
    const float2 b = make_float2(g.x > 0.f ? bA / g.x : 0.f, g.y > 0.f ? bE / g.y : 0.f);
    wb[k] = b;
    not_one += (g.x > 0.f && b.x != 1.0f) + (g.y > 0.f && b.y != 1.0f);
  }
  for (int i = threadIdx.x; i < n_valid; i += 1024) wa[i] = g;
  if (not_one) atomicAdd(&counts[1], not_one);
}

// Compacted list of valid (non-gap) tranches and its prefix counts (C10).  One block.  valid_m is padded to
// ncol_cap entries with its last entry (entry 0 = tranche 0 when everything is masked).
__global__ void __launch_bounds__(1024)
valid_list_kernel(const uint8_t* __restrict__ gap, int Nt, int ncol_cap, int* __restrict__ vprefix, int* __restrict__ valid_m) {
  __shared__ int s_cnt[1024];
  __shared__ int s_last;
  const int t = threadIdx.x;
  const int per = (Nt + 1023) / 1024;
  const int b = min(t * per, Nt), e = min(b + per, Nt);
  int c = 0;
  for (int m = b; m < e; ++m) c += gap[m] != 0;
  s_cnt[t] = c;
  if (t == 0) s_last = 0;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {                           // inclusive Hillis-Steele scan
    const int v = t >= o ? s_cnt[t - o] : 0;
    __syncthreads();
    s_cnt[t] += v;
    __syncthreads();
  }
  int pos = s_cnt[t] - c;
  const int total = s_cnt[1023];
  for (int m = b; m < e; ++m) {
    vprefix[m] = pos;
    if (gap[m] != 0) {
      valid_m[pos++] = m;
      if (pos == total) s_last = m;
    }
  }
  if (t == 1023) vprefix[Nt] = total;
  __syncthreads();
  for (int i = total + t; i < ncol_cap; i += 1024) valid_m[i] = s_last;
}

// ------------------------------------------------------------------------------------------
// Measurement aid (bench.py): read an L2-resident buffer over and over with
// coalesced 16-byte loads from every SM; the resulting GB/s is the on-chip gather ceiling that the
// roofline's L2 term is quoted against.  The sums are written so the loads cannot be dropped.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024, 1)
l2_probe_kernel(const float4* __restrict__ buf, long long n_vec, int iters, float* __restrict__ sink) {
  float acc = 0.f;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (int it = 0; it < iters; ++it) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < n_vec; i += 4 * stride) {
      const float4 a = __ldcg(buf + i), b = __ldcg(buf + i + stride), c = __ldcg(buf + i + 2 * stride),
                   d = __ldcg(buf + i + 3 * stride);
      acc += (a.x + b.y) + (c.z + d.w);
    }
    for (; i < n_vec; i += stride) acc += __ldcg(buf + i).x;
  }
  if (acc == 123.456f) sink[0] = acc;      // never true for the zero-filled buffer; keeps the loads alive
}

// ------------------------------------------------------------------------------------------
// Ladder refinement (a10; C19): child (a, b) of survivor j, a, b in [0, r), sits at
//   Mc' = Mc (1 + o_a d_mc_rel),  tc' = tc + o_b d_tc,  o_i = (2i + 1 - r) / (2r)
// (an r x r lattice, r times denser per dimension, that tiles the parent's cell); the other six
// columns are copied.  One thread per child; products and sums are rounded separately (no FMA
// contraction) so the rows are bit-identical to an IEEE fp64 evaluation in the stated order.
// A parent index outside [0, n) gives a NaN row, which tfs_eval counts as a bad template.
// ------------------------------------------------------------------------------------------
__global__ void refine_kernel(const double* __restrict__ params, long long n, const long long* __restrict__ idx,
                              long long k, int r, double d_mc_rel, double d_tc, double* __restrict__ out) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long rr = (long long)r * r;
  if (t >= k * rr) return;
  const long long j = t / rr;
  const int ab = (int)(t - j * rr);
  const int ia = ab / r, ib = ab - ia * r;
  const long long src = idx[j];
  double* o = out + t * 8;
  if (src < 0 || src >= n) {
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
#pragma unroll
    for (int c = 0; c < 8; ++c) o[c] = qnan;
    return;
  }
  const double* p = params + src * 8;
  const double oa = __ddiv_rn((double)(2 * ia + 1 - r), (double)(2 * r));
  const double ob = __ddiv_rn((double)(2 * ib + 1 - r), (double)(2 * r));
  o[0] = __dmul_rn(p[0], __dadd_rn(1.0, __dmul_rn(oa, d_mc_rel)));
  o[1] = __dadd_rn(p[1], __dmul_rn(ob, d_tc));
#pragma unroll
  for (int c = 2; c < 8; ++c) o[c] = p[c];
}

// ------------------------------------------------------------------------------------------
// Tile search (P:275 tiles in (M_c, f_in), P:57 t_c = remaining lifetime at t_0 = 0).
// tau(f) = 5 M (8 pi M f)^(-8/3), f(tau) = (tau/5M)^(-3/8)/(8 pi M): the 0PN track of load_template/track_point
// solved for the time to coalescence.  Lattice positions are formed with separately rounded products and sums
// (bit-identical to the host arithmetic of the oracle); the two powers go through pow().
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double tau_of_f(double Mc, double f) {
  const double M = __dmul_rn(Mc, kMtsun);
  const double z = __dmul_rn(__dmul_rn(__dmul_rn(8.0, kPi), M), f);
  return __dmul_rn(__dmul_rn(5.0, M), pow(z, -8.0 / 3.0));
}
__device__ __forceinline__ double f_of_tau(double Mc, double tau) {
  const double M = __dmul_rn(Mc, kMtsun);
  return __ddiv_rn(pow(__ddiv_rn(tau, __dmul_rn(5.0, M)), -0.375), __dmul_rn(__dmul_rn(8.0, kPi), M));
}

struct Row8 { double v[8]; };

// cell-centred lattice over [mc_lo, mc_lo + n_mc d_mc] x [fin_lo, fin_lo + n_fin d_fin]; row i n_fin + j
__global__ void tile_lattice_kernel(double mc_lo, double d_mc, int n_mc, double fin_lo, double d_fin, int n_fin,
                                    const Row8 row, double* __restrict__ out) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)n_mc * n_fin) return;
  const int i = (int)(t / n_fin), j = (int)(t - (long long)i * n_fin);
  const double mc = __dadd_rn(mc_lo, __dmul_rn(__dadd_rn((double)i, 0.5), d_mc));
  const double fin = __dadd_rn(fin_lo, __dmul_rn(__dadd_rn((double)j, 0.5), d_fin));
  double* o = out + t * 8;
  o[0] = mc;
  o[1] = tau_of_f(mc, fin);
#pragma unroll
  for (int c = 2; c < 8; ++c) o[c] = row.v[c];
}

// r*r children per survivor in (M_c, f_in): M_c' = M_c + o_a d_mc, f_in' = f_in + o_b d_fin, t_c' = tau(M_c', f_in')
__global__ void refine_fin_kernel(const double* __restrict__ params, long long n, const long long* __restrict__ idx,
                                  long long k, int r, double d_mc, double d_fin, double* __restrict__ out) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long rr = (long long)r * r;
  if (t >= k * rr) return;
  const long long j = t / rr;
  const int ab = (int)(t - j * rr);
  const int ia = ab / r, ib = ab - ia * r;
  const long long src = idx[j];
  double* o = out + t * 8;
  if (src < 0 || src >= n) {
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
#pragma unroll
    for (int c = 0; c < 8; ++c) o[c] = qnan;
    return;
  }
  const double* p = params + src * 8;
  const double oa = __ddiv_rn((double)(2 * ia + 1 - r), (double)(2 * r));
  const double ob = __ddiv_rn((double)(2 * ib + 1 - r), (double)(2 * r));
  const double fin = f_of_tau(p[0], p[1]);
  const double mc = __dadd_rn(p[0], __dmul_rn(oa, d_mc));
  o[0] = mc;
  o[1] = tau_of_f(mc, __dadd_rn(fin, __dmul_rn(ob, d_fin)));
#pragma unroll
  for (int c = 2; c < 8; ++c) o[c] = p[c];
}

// ------------------------------------------------------------------------------------------
// Top-k: radix select on 64-bit composite keys (value order, then lower index), then bitonic sort.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long topk_key(float v, unsigned idx) {
  unsigned b = __float_as_uint(v);
  if (v == 0.0f) b = 0u;                                      // -0.0 ties with +0.0
  unsigned o = (b & 0x80000000u) ? ~b : (b | 0x80000000u);   // ascending unsigned == ascending float
  if (v != v) o = 0u;                                         // NaN below everything
  return ((unsigned long long)o << 32) | (unsigned long long)(0xFFFFFFFFu - idx);
}

struct SelectState {
  unsigned long long prefix;      // high bits fixed so far
  unsigned long long k_rem;       // rank still to find inside the prefix bucket
  unsigned hist[256];
  unsigned out_count;
};

__global__ void topk_init_kernel(SelectState* st, unsigned long long k) {
  if (threadIdx.x == 0) { st->prefix = 0; st->k_rem = k; st->out_count = 0; }
  if (threadIdx.x < 256) st->hist[threadIdx.x] = 0;
}

__global__ void topk_hist_kernel(const float* __restrict__ v, long long n, int pass, SelectState* st) {
  __shared__ unsigned sh[256];
  if (threadIdx.x < 256) sh[threadIdx.x] = 0;
  __syncthreads();
  const int shift = 56 - 8 * pass;
  const unsigned long long prefix = st->prefix;
  const unsigned long long himask = pass == 0 ? 0ULL : (~0ULL << (shift + 8));
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const unsigned long long key = topk_key(v[i], (unsigned)i);
    if ((key & himask) == prefix) atomicAdd(&sh[(unsigned)(key >> shift) & 255u], 1u);
  }
  __syncthreads();
  if (threadIdx.x < 256 && sh[threadIdx.x]) atomicAdd(&st->hist[threadIdx.x], sh[threadIdx.x]);
}

__global__ void topk_pick_kernel(int pass, SelectState* st) {
  // one thread: walk the histogram from the top digit down to the bucket holding rank k_rem
  if (threadIdx.x == 0) {
    unsigned long long k = st->k_rem;
    const int shift = 56 - 8 * pass;
    int d = 255;
    for (; d > 0; --d) {
      const unsigned c = st->hist[d];
      if (k <= c) break;
      k -= c;
    }
    st->k_rem = k;
    st->prefix |= ((unsigned long long)d << shift);
  }
  __syncthreads();
  if (threadIdx.x < 256) st->hist[threadIdx.x] = 0;
}

__global__ void topk_gather_kernel(const float* __restrict__ v, long long n, SelectState* st,
                                   unsigned long long* __restrict__ keys, unsigned cap) {
  const unsigned long long thr = st->prefix;          // exact key of the k-th largest element
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const unsigned long long key = topk_key(v[i], (unsigned)i);
    if (key >= thr) {
      const unsigned pos = atomicAdd(&st->out_count, 1u);
      if (pos < cap) keys[pos] = key;
    }
  }
}

__global__ void topk_pad_kernel(unsigned long long* keys, unsigned from, unsigned to) {
  const unsigned i = from + blockIdx.x * blockDim.x + threadIdx.x;
  if (i < to) keys[i] = 0ULL;
}

// one bitonic compare-exchange step over P keys (descending overall)
__global__ void bitonic_step_kernel(unsigned long long* keys, unsigned P, unsigned size, unsigned stride) {
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= P / 2) return;
  const unsigned lo = 2 * stride * (t / stride) + (t % stride);
  const unsigned hi = lo + stride;
  const bool desc = ((lo & size) == 0);
  const unsigned long long a = keys[lo], b = keys[hi];
  if ((a < b) == desc) { keys[lo] = b; keys[hi] = a; }
}

// whole sort in shared memory when P <= 4096
__global__ void bitonic_small_kernel(unsigned long long* keys, unsigned P) {
  extern __shared__ unsigned long long sk[];
  for (unsigned i = threadIdx.x; i < P; i += blockDim.x) sk[i] = keys[i];
  __syncthreads();
  for (unsigned size = 2; size <= P; size <<= 1) {
    for (unsigned stride = size >> 1; stride > 0; stride >>= 1) {
      for (unsigned t = threadIdx.x; t < P / 2; t += blockDim.x) {
        const unsigned lo = 2 * stride * (t / stride) + (t % stride);
        const unsigned hi = lo + stride;
        const bool desc = ((lo & size) == 0);
        const unsigned long long a = sk[lo], b = sk[hi];
        if ((a < b) == desc) { sk[lo] = b; sk[hi] = a; }
      }
      __syncthreads();
    }
  }
  for (unsigned i = threadIdx.x; i < P; i += blockDim.x) keys[i] = sk[i];
}

// P > 4096: each block owns kBitonicBlock consecutive keys in shared memory and runs every compare-exchange
// step whose stride stays inside the block (stride <= kBitonicBlock/2) for the sizes size_first ... size_last;
// the few steps with a larger stride run in bitonic_step_kernel.  Directions use the global index.
constexpr unsigned kBitonicBlock = 4096;
__global__ void __launch_bounds__(1024)
bitonic_block_kernel(unsigned long long* keys, unsigned size_first, unsigned size_last) {
  __shared__ unsigned long long sk[kBitonicBlock];
  const unsigned base = blockIdx.x * kBitonicBlock;
  for (unsigned i = threadIdx.x; i < kBitonicBlock; i += blockDim.x) sk[i] = keys[base + i];
  __syncthreads();
  for (unsigned size = size_first; size <= size_last && size != 0; size <<= 1) {
    for (unsigned stride = min(size >> 1, kBitonicBlock / 2); stride > 0; stride >>= 1) {
      for (unsigned t = threadIdx.x; t < kBitonicBlock / 2; t += blockDim.x) {
        const unsigned lo = 2 * stride * (t / stride) + (t % stride);
        const unsigned hi = lo + stride;
        const bool desc = (((base + lo) & size) == 0);
        const unsigned long long a = sk[lo], b = sk[hi];
        if ((a < b) == desc) { sk[lo] = b; sk[hi] = a; }
      }
      __syncthreads();
    }
  }
  for (unsigned i = threadIdx.x; i < kBitonicBlock; i += blockDim.x) keys[base + i] = sk[i];
}

// Small batches (n <= kBitonicBlock, e.g. the 64-template batches of BASELINE.json configs[0]): the whole select in ONE
// launch -- keys of all n values into shared memory (padding keys are 0: below every real key, whose low word is
// 0xFFFFFFFF - idx > 0 for idx < 2^32 - 1), bitonic sort descending, emit the first k.  Same order as the general path.
__global__ void __launch_bounds__(1024)
topk_small_kernel(const float* __restrict__ v, int n, int k, long long* __restrict__ idx, float* __restrict__ val) {
  __shared__ unsigned long long sk[kBitonicBlock];
  unsigned P = 2;
  while (P < (unsigned)n) P <<= 1;
  for (unsigned i = threadIdx.x; i < P; i += blockDim.x) sk[i] = i < (unsigned)n ? topk_key(v[i], i) : 0ULL;
  __syncthreads();
  for (unsigned size = 2; size <= P; size <<= 1) {
    for (unsigned stride = size >> 1; stride > 0; stride >>= 1) {
      for (unsigned t = threadIdx.x; t < P / 2; t += blockDim.x) {
        const unsigned lo = 2 * stride * (t / stride) + (t % stride);
        const unsigned hi = lo + stride;
        const bool desc = ((lo & size) == 0);
        const unsigned long long a = sk[lo], b = sk[hi];
        if ((a < b) == desc) { sk[lo] = b; sk[hi] = a; }
      }
      __syncthreads();
    }
  }
  for (unsigned i = threadIdx.x; i < (unsigned)k; i += blockDim.x) {
    const unsigned id = 0xFFFFFFFFu - (unsigned)(sk[i] & 0xFFFFFFFFull);
    idx[i] = (long long)id;
    val[i] = v[id];
  }
}

__global__ void topk_emit_kernel(const unsigned long long* __restrict__ keys, const float* __restrict__ v,
                                 int k, long long* __restrict__ idx, float* __restrict__ val) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= k) return;
  const unsigned id = 0xFFFFFFFFu - (unsigned)(keys[i] & 0xFFFFFFFFull);
  idx[i] = (long long)id;
  val[i] = v[id];
}

}  // namespace tfs
