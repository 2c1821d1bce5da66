// tfs_kernels.cuh -- device code of libtfs (sm_100a).  See include/tfs.h for the operation and
// DESIGN.md section 6 for the kernel design.  Citations: P:<line> of PAPER.md, C<n> = DESIGN.md.
//
// Work decomposition: one WARP evaluates one (template, time tile) pair.  A time tile is a run
// of kTileMax consecutive VALID (non-gap) tranches, whatever N_seg is; work items are ordered
// tile-major so that all templates sweep the same slab of the grid together and the slab stays
// L2-resident.  Segment boundaries cut a tile into PIECES; the warp writes one partial per piece.
// Inside a tile lanes are tranches (32 at a time): fp64 0PN track per lane, then each lane walks
// its own window; the grid is stored time-contiguous so those loads coalesce across lanes.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tfs {

// Warps of the one persistent CTA per SM.  The kernel is short of warps to hide its dependent chains, so
// it runs the most a CTA can hold: 32 warps at 64 registers per thread (measured against 20, 24, 26, 28
// for both the separable- and the general-weights variants).
#ifndef TFS_WARPS_SEPARABLE
#define TFS_WARPS_SEPARABLE 32
#endif
#ifndef TFS_WARPS_GENERAL
#define TFS_WARPS_GENERAL 32
#endif
constexpr int kMaxWarpsPerCta = TFS_WARPS_SEPARABLE > TFS_WARPS_GENERAL ? TFS_WARPS_SEPARABLE : TFS_WARPS_GENERAL;
#ifndef TFS_TILE
#define TFS_TILE 512
#endif
constexpr int kTileMax = TFS_TILE;       // valid tranches per time tile (16 chunks of 32 lanes)
constexpr int kLutN = 512;          // LUT intervals in t = 1/(1+v)
constexpr double kMtsun = 4.925490947e-6;   // G Msun / c^3 [s]
constexpr double kPi = 3.14159265358979323846;

// f(v) = w (F0 + F1 w^4 + F2 w^8), g(v) = w^3 (G0 + G1 w^4 + G2 w^8), w = 1/v, valid for |v| >= kVFar
struct FarCoef { float F0, F1, F2, G0, G1, G2; };

struct EvalArgs {
  const float4* __restrict__ grid;     // [Nf][Nt] (time-contiguous) {Y_A.re, Y_E.re, Y_A.im, Y_E.im}, Y = W*D
  const float2* __restrict__ wgt;      // [Nf][Nt] {W_A, W_E}
  const float2* __restrict__ wa;       // [Nt] {a_A, a_E}  (separable weights: W = a[m] b[k])
  const float2* __restrict__ wb;       // [Nf + kPadRows] {b_A, b_E}
  const uint8_t* __restrict__ gap;     // [Nt] 1 = valid
  const int* __restrict__ vprefix;     // [Nt+1] number of valid tranches before m
  const int* __restrict__ valid_m;     // [vprefix[Nt]] the valid tranche indices, ascending (padded to >= 1 entry)
  const int* __restrict__ tile_first;  // [n_tiles+1] first piece of each tile (pieces are numbered in time order)
  const int* __restrict__ piece_end;   // [n_pieces] entry of valid_m where the piece ends (exclusive)
  const float4* __restrict__ lut;      // [kLutN+1] {a_G, a_F, b_G, b_F} (see fresnel_aux)
  const double* __restrict__ params;   // [n][8]
  float4* __restrict__ partials;       // [n_pieces][n] {z.re, z.im, hh, 0}
  unsigned long long* bad_count;       // templates rejected (counted on tile 0 only)
  unsigned long long* work_counter;    // next unclaimed work item (zeroed before each launch)
  long long n;                         // templates in this launch
  int Nt, Nf;
  int n_valid, n_tiles;                // valid tranches, ceil(n_valid / kTileMax) (>= 1)
  int H, adaptive;
  double DT;
  double x_lo, x_hi;                   // band in bins: f_lo*DT, f_hi*DT
  double c_max;
  FarCoef far;                         // far-zone polynomials of f, g (fitted at tfs_create)
};

// Per-template constants derived from the parameter row.
struct TemplateConst {
  double tc, phic_turns, inv5M;
  double xcoefDT;        // DT / (8 pi M):           x = f DT = X^{-3/8} xcoefDT
  double ccoef;          // (3/8) DT / (5M):         c = fdot DT^2 = x ccoef / X
  float acoef;           // amp (8 pi M)^{-2/3}:     A_m = acoef X^{-1/4}
  double TAr, TAi, TEr, TEi;
  bool ok;
};

__device__ __forceinline__ TemplateConst load_template(const double* __restrict__ p, double DT) {
  TemplateConst t;
  const double Mc = p[0];
  t.tc = p[1];
  const double phic = p[2];
  t.TAr = p[3]; t.TAi = p[4]; t.TEr = p[5]; t.TEi = p[6];
  const double amp = p[7];
  bool ok = isfinite(Mc) && isfinite(t.tc) && isfinite(phic) && isfinite(t.TAr) && isfinite(t.TAi) &&
            isfinite(t.TEr) && isfinite(t.TEi) && isfinite(amp) && (Mc > 0.0);
  const double M = (ok ? Mc : 1.0) * kMtsun;
  t.inv5M = 1.0 / (5.0 * M);
  const double xcoef = 1.0 / (8.0 * kPi * M);                // f = X^{-3/8} xcoef
  t.xcoefDT = xcoef * DT;
  t.ccoef = 0.375 * DT * t.inv5M;
  // A_m = amp f^{2/3} = amp xcoef^{2/3} X^{-1/4}; a common factor of the template (fp32 is enough)
  const float cx = cbrtf((float)xcoef);
  t.acoef = (float)(ok ? amp : 0.0) * cx * cx;
  t.phic_turns = (ok ? phic : 0.0) * (0.5 / kPi);
  t.ok = ok;
  return t;
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
__device__ __forceinline__ TrackPoint track_point(const TemplateConst& t, int m, double DT,
                                                  double x_lo, double x_hi, double c_max, bool valid) {
  TrackPoint r;
  const double tau = t.tc - (double)m * DT;
  bool act = valid && (tau > DT);
  const double X = act ? tau * t.inv5M : 1.0;
  double y0 = (double)exp2f(-0.125f * __log2f((float)X));
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
  act = act && (r.x >= x_lo) && (r.x + r.c <= x_hi) && (r.c <= c_max);
  r.active = act;
  return r;
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
// In shared memory it is stored kLutCopies times, copy r of entry i at 16-byte slot
// (i*kLutCopies + r), and lane l reads copy l & 7: the 8 lanes of a quarter-warp always hit 8
// different bank groups, so an LDS.128 is conflict-free whatever the indices are.
constexpr int kLutCopies = 8;
constexpr float kMagic = 12582912.0f;          // 1.5 * 2^23: (p + kMagic) rounds p to an integer in the mantissa
constexpr unsigned kMagicBits = 0x4B400000u;

__device__ __forceinline__ float rcp_approx(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

__device__ __forceinline__ float4 lds128(unsigned addr) {
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
// lut_lane = shared address of this lane's LUT copy minus kMagicBits * (16 * kLutCopies)  (mod 2^32).
template <int MODE>
__device__ __forceinline__ void fresnel_aux(float v, unsigned lut_lane, f2_t& GF, float& ts) {
  const float a = fabsf(v);
  if (MODE == 0) {
    const float t = rcp_approx(1.0f + a);         // MUFU.RCP
    const float q = fmaf(t, (float)kLutN, kMagic);
    const float4 e = lds128(__float_as_uint(q) * (16u * kLutCopies) + lut_lane);   // {a_G, a_F, b_G, b_F}
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

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// dynamic shared memory of kernel A: [LUT copies][per-lane tile sums: 3 packed pairs per thread, stored [3][threads]]
constexpr int kLutSmemBytes = (kLutN + 1) * kLutCopies * (int)sizeof(float4);
constexpr int kEvalSmemBytes = kLutSmemBytes + 3 * kMaxWarpsPerCta * 32 * (int)sizeof(f2_t);

// One pixel of one tranche (a3-a5).  The template coefficient is h = P h', P = A/sqrt(2c) exp(i phi_m)
// constant over the tranche, and (auxiliary-function form of Eq. 16)
//   h' = Godd(v0) - Godd(v1) E  [+ (1+i) exp(-i pi u^2/c) inside the swept band],
//   Godd(v) = sign(v) (g(|v|) + i f(|v|)),  E = exp(i psi), psi = pi c + 2 pi frac(x).
// The loop accumulates z'_alpha += conj(Y_alpha) h', q'_alpha += W_alpha |h'|^2 and the factor P
// (|P|^2 for q) is applied once per tranche.
//
// Two evaluations of Godd:
//   FAR  (|v0|, |v1| >= kVFar):  f(v) = w Pf(w^4), g(v) = w^3 Pg(w^4), w = 1/v, Pf and Pg quadratics
//         fitted at tfs_create (they are the asymptotic series of A&S 7.3.27-28 re-fitted on the
//         interval; odd in v, so the sign comes for free).  No table read: 2 MUFU.RCP + 10 packed ops.
//   NEAR (anything else): the shared-memory LUT in t = 1/(1+|v|) (fresnel_aux).
// The far zone covers all but the ~2 pixels next to the track for the slow chirps that make up the
// bulk of every bank (|v| = sqrt(2/c) |u|).
constexpr float kVFar = 3.0f;


struct LaneTrack {      // per-lane (= per-tranche) constants of the pixel loop
  float sc;             // sqrt(2/c)
  float kap;            // sqrt(c/2) = 1/sc
  float c;              // v1 - v0 = sc * c
  float hc;             // 1/(2c): pi u^2/c = 2 pi (u^2 hc)
  float Er, Ei;         // exp(i psi)
};

struct LaneSums { f2_t zr, zi, q; };     // {A, E} pairs: Re z', Im z', q'

// Weight modes (chosen by tfs_upload_data, C11):
//   kWGeneral    per-pixel weights W[alpha,m,k], read next to every data pixel
//   kWSeparable  W[alpha,m,k] = a_alpha[m] b_alpha[k]: b from a small [Nf] table, a applied once per tranche
//   kWTimeOnly   b = 1: no weight is read in the pixel loop, q' = sum |h'|^2 for both channels
constexpr int kWGeneral = 0, kWSeparable = 1, kWTimeOnly = 2;

// grid pixel Y = {Y_A.re, Y_E.re, Y_A.im, Y_E.im}, weights Wt = {W_A, W_E} (or {b_A, b_E})
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

template <int MODE, int MASKED>
__device__ __forceinline__ void pixel_near(const LaneTrack& L, float u, float msk, unsigned lut_lane,
                                           float& hr, float& hi) {
  const float v0 = L.sc * u;
  const float v1 = fmaf(L.sc, L.c, v0);
  f2_t GF0, GF1;
  float t0, t1;
  fresnel_aux<MODE>(v0, lut_lane, GF0, t0);
  fresnel_aux<MODE>(v1, lut_lane, GF1, t1);
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
}

// Pixel loop of one chunk (32 tranches, one per lane): every lane walks its own window, offsets
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
#ifndef TFS_GROUP
#define TFS_GROUP 2
#endif
constexpr int kGroup = TFS_GROUP;
constexpr int kPadRows = 16;                 // rows of zero padding behind the grid and the weights
constexpr int kRagMax = kPadRows - 2 * kGroup;   // largest Wmax - Wmin handled without clamping the loads
static_assert(kRagMax >= 1, "kPadRows too small for kGroup");

// ZONES: 1 = test the offset against the near zone, 0 = the offset is known to be far
template <int MODE, int WMODE, int MASKED, int ZONES>
__device__ __forceinline__ void pixel_step(const LaneTrack& L, const FarCoef& C, int jj, int Wm, int JA, int JB,
                                           const float4 Yc, const float2 Wc, float& u, unsigned lut_lane,
                                           LaneSums& s) {
  const float msk = (MASKED && jj >= Wm) ? 0.0f : 1.0f;
  float hr, hi;
  if (ZONES && jj >= JA && jj < JB) pixel_near<MODE, MASKED>(L, u, msk, lut_lane, hr, hi);
  else pixel_far<MASKED>(L, C, u, msk, hr, hi);
  mac<WMODE>(s, Yc, Wc, hr, hi);
  u -= 1.0f;
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
    if (i < 0 || i >= (a.Nf + TFS_BOUNDS_PAD) * a.Nt || kb + jj * kstp < 0 || kb + jj * kstp >= a.Nf + TFS_BOUNDS_PAD) __trap();
#endif
    B.Y[p] = __ldg(a.grid + i);
    if (WMODE == kWGeneral) B.W[p] = __ldg(a.wgt + i);
    if (WMODE == kWSeparable) B.W[p] = __ldg(a.wb + kb + jj * kstp);
  }
}

template <int MODE, int WMODE, int MASKED>
__device__ __forceinline__ void compute_group(const LaneTrack& L, const FarCoef& C, const PixelBuf& B, int j0, int Wm,
                                              int Wmax, int JA, int JB, float& u, unsigned lut_lane, LaneSums& s) {
  if (j0 < JB && j0 + kGroup > JA) {
#pragma unroll
    for (int p = 0; p < kGroup; ++p)
      if (!MASKED || j0 + p < Wmax)
        pixel_step<MODE, WMODE, MASKED, 1>(L, C, j0 + p, Wm, JA, JB, B.Y[p], B.W[p], u, lut_lane, s);
  } else {
#pragma unroll
    for (int p = 0; p < kGroup; ++p)
      if (!MASKED || j0 + p < Wmax)
        pixel_step<MODE, WMODE, MASKED, 0>(L, C, j0 + p, Wm, JA, JB, B.Y[p], B.W[p], u, lut_lane, s);
  }
}

// one group from buffer B: unmasked while the whole group lies below Wmin
template <int MODE, int WMODE>
__device__ __forceinline__ void compute_group_auto(const LaneTrack& L, const FarCoef& C, const PixelBuf& B, int j0,
                                                   int Wm, int Wmin, int Wmax, int JA, int JB, float& u,
                                                   unsigned lut_lane, LaneSums& s) {
  if (j0 + kGroup <= Wmin) compute_group<MODE, WMODE, 0>(L, C, B, j0, Wm, Wmax, JA, JB, u, lut_lane, s);
  else compute_group<MODE, WMODE, 1>(L, C, B, j0, Wm, Wmax, JA, JB, u, lut_lane, s);
}

// idx = pixel index of offset 0, stp = Nt for an active lane and 0 otherwise, Wm = window length (>= 1
// for active lanes, 0 otherwise)
template <int MODE, int WMODE>
__device__ __forceinline__ void pixel_loop(const EvalArgs& a, const LaneTrack& L, const FarCoef& C, int Wm, int Wmin,
                                           int Wmax, int JA, int JB, int idx, int stp, int kb, int kstp, float u,
                                           unsigned lut_lane, LaneSums& s) {
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
      compute_group_auto<MODE, WMODE>(L, C, A, j, Wm, Wmin, Wmax, JA, JB, u, lut_lane, s);
      if (j + kGroup >= Wmax) break;
      if (j + 2 * kGroup < Wmax) load_group<0, WMODE>(a, A, idx, stp, kb, kstp, j + 2 * kGroup, jlast);
      compute_group_auto<MODE, WMODE>(L, C, B, j + kGroup, Wm, Wmin, Wmax, JA, JB, u, lut_lane, s);
    }
  } else {
    // very ragged chunk (wide tracks next to narrow ones): every load clamped, every step masked
    load_group<1, WMODE>(a, A, idx, stp, kb, kstp, 0, jlast);
    for (int j = 0; j < Wmax; j += 2 * kGroup) {
      load_group<1, WMODE>(a, B, idx, stp, kb, kstp, j + kGroup, jlast);
      compute_group<MODE, WMODE, 1>(L, C, A, j, Wm, Wmax, JA, JB, u, lut_lane, s);
      if (j + kGroup >= Wmax) break;
      load_group<1, WMODE>(a, A, idx, stp, kb, kstp, j + 2 * kGroup, jlast);
      compute_group<MODE, WMODE, 1>(L, C, B, j + kGroup, Wm, Wmax, JA, JB, u, lut_lane, s);
    }
  }
}

// ------------------------------------------------------------------------------------------
// Kernel A: track + gather + per-tile sums.  Persistent: one CTA per SM, warps claim work items
// (template, tile) in tile-major order from a global counter, kClaim at a time.
// Inside a work item LANES ARE TRANCHES: lane l owns the l-th valid (non-gap) tranche of the
// current chunk of 32, computes its track point in fp64 and then walks its own window pixel by
// pixel.  The grid is stored time-contiguous ([k][m]), so the 32 lanes' loads of pixel offset j
// fall on consecutive addresses wherever neighbouring tranches share k_lo (slow chirps: runs of
// 1/c tranches).  Per chunk the window offsets are split (warp-uniformly) into the NEAR zone around
// the track, evaluated from the shared-memory LUT, and the FAR zone, evaluated from the fitted
// asymptotic polynomials in packed fp32 (pixel_loop).
// ------------------------------------------------------------------------------------------
constexpr int kClaim = 4;

// Piece table (C9, C10).  Segment n = tranches [ceil(n Nt/N_seg), ceil((n+1) Nt/N_seg)), i.e. n(m) =
// floor(m N_seg / Nt).  Tile t = entries [t kTileMax, (t+1) kTileMax) of the compacted valid-tranche list.
// A piece is a maximal run of entries inside one tile and one segment; pieces are numbered in time order.
// One thread walks the list (<= n_tiles + N_seg pieces); the table is cached per N_seg by the host.
//   tile_first[t] = first piece of tile t, tile_first[n_tiles] = number of pieces
//   piece_end[p]  = entry where piece p ends (exclusive);  piece_seg[p] = its segment
__global__ void piece_table_kernel(const int* __restrict__ vprefix, const int* __restrict__ valid_m, int Nt, int N_seg,
                                   int n_valid, int n_tiles, int* __restrict__ tile_first,
                                   int* __restrict__ piece_end, int* __restrict__ piece_seg) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  int p = 0;
  for (int t = 0; t < n_tiles; ++t) {
    tile_first[t] = p;
    int i = t * kTileMax;
    const int iend = min(i + kTileMax, n_valid);
    while (i < iend) {
      const int seg = (int)(((long long)valid_m[i] * N_seg) / Nt);
      const int s1 = (int)(((long long)(seg + 1) * Nt + N_seg - 1) / N_seg);     // first tranche of the next segment
      const int e = min(vprefix[min(s1, Nt)], iend);
      piece_seg[p] = seg;
      piece_end[p] = e;
      ++p;
      i = e;
    }
  }
  tile_first[n_tiles] = p;
}

__host__ __device__ constexpr int warps_per_cta(int wmode) {
  return wmode == 0 ? TFS_WARPS_GENERAL : TFS_WARPS_SEPARABLE;      // 0 = kWGeneral (declared below)
}

template <int MODE, int WMODE>
__global__ void __launch_bounds__(warps_per_cta(WMODE) * 32, 1)
eval_tiles_kernel(const EvalArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* s_lut = reinterpret_cast<float4*>(smem_raw);
  f2_t* s_acc = reinterpret_cast<f2_t*>(smem_raw + kLutSmemBytes) + threadIdx.x;       // [3][blockDim]
  constexpr int kAccStride = warps_per_cta(WMODE) * 32;

  const int lane = threadIdx.x & 31;
  if (MODE == 0) {
    for (int i = threadIdx.x; i < (kLutN + 1) * kLutCopies; i += blockDim.x) s_lut[i] = a.lut[i / kLutCopies];
    __syncthreads();
  }
  const unsigned lut_lane = (unsigned)__cvta_generic_to_shared(s_lut) + 16u * (unsigned)(lane & (kLutCopies - 1)) -
                            kMagicBits * (16u * kLutCopies);

  const long long n_work = a.n * (long long)a.n_tiles;
  for (;;) {
    long long w0 = 0;
    if (lane == 0) w0 = (long long)atomicAdd(a.work_counter, (unsigned long long)kClaim);
    w0 = __shfl_sync(0xffffffffu, w0, 0);
    if (w0 >= n_work) break;
    const int n_claim = (int)min((long long)kClaim, n_work - w0);
    int tile = (int)(w0 / a.n);
    long long it = w0 - (long long)tile * a.n;
    for (int wi = 0; wi < n_claim; ++wi, ++it) {
      if (it == a.n) { it = 0; ++tile; }
      // valid (non-gap) tranches of the tile: entries [i0, i1) of the compacted list (C10), cut by the
      // segment boundaries into pieces [p, p_last]
      const int i0 = tile * kTileMax, i1 = min(i0 + kTileMax, a.n_valid);
      int p = a.tile_first[tile];
      const int p_stop = a.tile_first[tile + 1];

      const TemplateConst T = load_template(a.params + it * 8, a.DT);
      if (!T.ok) {
        for (int q = p + lane; q < p_stop; q += 32) a.partials[(long long)q * a.n + it] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (lane == 0 && tile == 0) atomicAdd(a.bad_count, 1ULL);
        continue;
      }
      int pend = p < p_stop ? a.piece_end[p] : i1;

      // per-lane running sums over the current piece ({A, E} pairs of Re z, Im z, q; <= kTileMax/32 chunk sums
      // each, fp32) live in shared memory; lanes, pieces and segments are then summed in fp64
#pragma unroll
      for (int v = 0; v < 3; ++v) s_acc[v * kAccStride] = pk(0.f, 0.f);

      // close piece p: sum its per-lane sums over the warp (packed fp32 butterfly: 32 terms), combine the
      // channels in fp64, store, reset
      auto flush = [&]() {
        f2_t r0 = s_acc[0 * kAccStride], r1 = s_acc[1 * kAccStride], r2 = s_acc[2 * kAccStride];
#pragma unroll
        for (int v = 0; v < 3; ++v) s_acc[v * kAccStride] = pk(0.f, 0.f);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          r0 = fadd2(r0, __shfl_xor_sync(0xffffffffu, r0, o));
          r1 = fadd2(r1, __shfl_xor_sync(0xffffffffu, r1, o));
          r2 = fadd2(r2, __shfl_xor_sync(0xffffffffu, r2, o));
        }
        if (lane == 0) {
          float zAr, zEr, zAi, zEi, qA, qE;
          upk(r0, zAr, zEr); upk(r1, zAi, zEi); upk(r2, qA, qE);
          const double dzAr = zAr, dzAi = zAi, dzEr = zEr, dzEi = zEi, dqA = qA, dqE = qE;
          // z = T_A z_A + T_E z_E ; hh = |T_A|^2 q_A + |T_E|^2 q_E   (Eq. 29, Eq. 31)
          const double zr = T.TAr * dzAr - T.TAi * dzAi + T.TEr * dzEr - T.TEi * dzEi;
          const double zi = T.TAr * dzAi + T.TAi * dzAr + T.TEr * dzEi + T.TEi * dzEr;
          const double hh = (T.TAr * T.TAr + T.TAi * T.TAi) * dqA + (T.TEr * T.TEr + T.TEi * T.TEi) * dqE;
          a.partials[(long long)p * a.n + it] = make_float4((float)zr, (float)zi, (float)hh, 0.f);
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
        f2_t vr = pk(0.f, 0.f), vi = vr, vq = vr;          // this chunk's per-lane contribution (P z', |P|^2 a q')
        if (act_mask != 0u) {
        int Wm = 0, idx = m, stp = 0, kb = 0, kstp = 0, ja = 0x7fffffff, jb = 0;
        float u = -1.f, Pr = 0.f, Pi = 0.f;
        LaneTrack L;        // inactive lanes: u_j = -1 - j, u_j + c = -0.5 - j (finite h' on zeroed data)
        L.sc = 1.f; L.kap = 1.f; L.c = 0.5f; L.hc = 0.f; L.Er = 0.f; L.Ei = 0.f;
        if (tp.active) {
          int k_lo, k_hi;
          window(tp, a.H, a.adaptive, a.Nf, k_lo, k_hi);
          Wm = k_hi - k_lo + 1;
          idx = k_lo * a.Nt + m;
          stp = a.Nt;
          kb = k_lo;
          kstp = 1;
          const double flx = floor(tp.x);
          const float fracx = (float)(tp.x - flx);
          u = fracx - (float)(k_lo - (int)flx);          // cancellation-safe x - k_lo
          // phases in turns, reduced in fp64 (phi reaches ~1e8 rad), then to [-1/2, 1/2)
          double tphi = T.phic_turns - tp.X58 * (1.0 / kPi);
          tphi -= floor(tphi);
          double tpsi = 0.5 * tp.c + (tp.x - flx);
          tpsi -= floor(tpsi);
          float sphi, cphi, spsi, cpsi;
          __sincosf(6.283185307179586f * ((float)tphi - 0.5f), &sphi, &cphi);     // = -(sin, cos)(2 pi tphi)
          __sincosf(6.283185307179586f * ((float)tpsi - 0.5f), &spsi, &cpsi);
          const float cf = (float)tp.c;
          L.sc = rsqrtf(0.5f * cf);
          L.kap = 0.5f * cf * L.sc;                                               // sqrt(c/2)
          L.c = cf;
          L.hc = __fdividef(0.5f, cf);
          const float pre = -(T.acoef * tp.Xm14) * (0.5f * L.sc);               // -A_m / sqrt(2c)
          Pr = pre * cphi;
          Pi = pre * sphi;
          L.Er = -cpsi;
          L.Ei = -spsi;
          // near zone of this lane: offsets j with |v0| < kVFar or |v1| < kVFar, i.e. -(c + d) < u - j < d
          const float d = fmaf(kVFar, L.kap, 1e-3f);
          ja = max((int)floorf(u - d) + 1, 0);
          jb = (int)ceilf(u + cf + d);
        }
        const int Wmax = __reduce_max_sync(0xffffffffu, Wm);
        const int Wmin = __reduce_min_sync(0xffffffffu, tp.active ? Wm : 0x7fffffff);
        int JA = __reduce_min_sync(0xffffffffu, ja);
        int JB = min(__reduce_max_sync(0xffffffffu, jb), Wmax);
        if (MODE != 0) { JA = 0; JB = Wmax; }          // the paper's approximants are used for every pixel
        JA = min(JA, JB);

        // ---------------- pixel loop (a3-a5): lane walks its own window ----------------
        LaneSums s;
        s.zr = pk(0.f, 0.f); s.zi = pk(0.f, 0.f); s.q = pk(0.f, 0.f);
        pixel_loop<MODE, WMODE>(a, L, a.far, Wm, Wmin, Wmax, JA, JB, idx, stp, kb, kstp, u, lut_lane, s);
        // apply the tranche's factor P to z' and |P|^2 (times a[m] for separable weights) to q'
        const float P2 = fmaf(Pr, Pr, Pi * Pi);
        f2_t qs = s.q, qc = pk(P2, P2);
        if (WMODE != kWGeneral) {
          // W = a[m] b[k]: the pixel loop summed b |h'|^2 (b = 1: {sum hr^2, sum hi^2})
          const float2 am = __ldg(a.wa + m);
          qc = pk(P2 * am.x, P2 * am.y);
          if (WMODE == kWTimeOnly) {
            float q0, q1;
            upk(s.q, q0, q1);
            qs = pk(q0 + q1, q0 + q1);
          }
        }
        if (!closes) {
          // the usual case: the whole chunk belongs to the current piece
          f2_t accr = s_acc[0 * kAccStride], acci = s_acc[1 * kAccStride];
          accr = ffma2(pk(Pr, Pr), s.zr, accr);          // Re (P z') = Pr zr - Pi zi
          accr = ffma2(pk(-Pi, -Pi), s.zi, accr);
          acci = ffma2(pk(Pr, Pr), s.zi, acci);          // Im (P z') = Pr zi + Pi zr
          acci = ffma2(pk(Pi, Pi), s.zr, acci);
          s_acc[0 * kAccStride] = accr;
          s_acc[1 * kAccStride] = acci;
          s_acc[2 * kAccStride] = ffma2(qc, qs, s_acc[2 * kAccStride]);
        } else {
          vr = fmul2(pk(Pr, Pr), s.zr);
          vr = ffma2(pk(-Pi, -Pi), s.zi, vr);
          vi = fmul2(pk(Pr, Pr), s.zi);
          vi = ffma2(pk(Pi, Pi), s.zr, vi);
          vq = fmul2(qc, qs);
        }
        }
        if (closes) {
          // every piece that ends inside this chunk (a segment boundary, or the end of the tile) takes the
          // lanes before its end and is closed; the lanes behind the last such end open the next piece
          int lo = 0;
          for (;;) {
            const bool ends = p < p_stop && pend <= cend;
            const int hi = ends ? pend - ic : 32;
            if (lane >= lo && lane < hi) {
              s_acc[0 * kAccStride] = fadd2(s_acc[0 * kAccStride], vr);
              s_acc[1 * kAccStride] = fadd2(s_acc[1 * kAccStride], vi);
              s_acc[2 * kAccStride] = fadd2(s_acc[2 * kAccStride], vq);
            }
            if (!ends) break;
            flush();
            ++p;
            if (p < p_stop) pend = a.piece_end[p];
            lo = hi;
          }
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// Kernel B: sum the piece partials of each segment, P_n = |z_n|^2/hh_n, Upsilon = sum_n P_n (Eq. 8, 9).
// Pieces are in time order, so the pieces of a segment are consecutive; a segment without a valid
// tranche has no piece and contributes 0.
// ------------------------------------------------------------------------------------------
__global__ void combine_kernel(const float4* __restrict__ partials, long long n, int N_seg,
                               const int* __restrict__ tile_first, int n_tiles, const int* __restrict__ piece_seg,
                               float* __restrict__ upsilon, float* __restrict__ seg_power,
                               float* __restrict__ seg_dh, float* __restrict__ seg_hh) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int n_pieces = tile_first[n_tiles];
  double ups = 0.0;
  int p = 0;
  for (int s = 0; s < N_seg; ++s) {
    double zr = 0, zi = 0, hh = 0;
    for (; p < n_pieces && piece_seg[p] == s; ++p) {
      const float4 v = partials[(long long)p * n + i];
      zr += v.x; zi += v.y; hh += v.z;
    }
    const double P = hh > 0.0 ? (zr * zr + zi * zi) / hh : 0.0;
    ups += P;
    if (seg_power) seg_power[i * N_seg + s] = (float)P;
    if (seg_dh) { seg_dh[(i * N_seg + s) * 2] = (float)zr; seg_dh[(i * N_seg + s) * 2 + 1] = (float)zi; }
    if (seg_hh) seg_hh[i * N_seg + s] = (float)hh;
  }
  upsilon[i] = (float)ups;
}

// ------------------------------------------------------------------------------------------
// Window pixel counts (phase 1 only).
// ------------------------------------------------------------------------------------------
__global__ void count_pixels_kernel(const EvalArgs a, long long* __restrict__ counts) {
  const int lane = threadIdx.x & 31;
  const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= a.n) return;
  const TemplateConst T = load_template(a.params + w * 8, a.DT);
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
// Upload (a0): Y = W*D interleaved by channel and W interleaved, transposed to time-contiguous
// [k][m] through a 32x32 shared-memory tile (reads coalesced along k, writes coalesced along m).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
pack_kernel(const float2* __restrict__ coeff, const float* __restrict__ weight, int Nt, int Nf,
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
      float2 dA = coeff[i], dE = coeff[npix + i];
      float wA = weight ? weight[i] : 1.0f;
      float wE = weight ? weight[npix + i] : 1.0f;
      // a pixel whose product W*D is not finite carries no information: weight 0 (also keeps every
      // value the gather can read finite, which pixel_loop relies on)
      if (!(isfinite(wA * dA.x) && isfinite(wA * dA.y) && isfinite(wA))) { wA = 0.f; dA = make_float2(0.f, 0.f); }
      if (!(isfinite(wE * dE.x) && isfinite(wE * dE.y) && isfinite(wE))) { wE = 0.f; dE = make_float2(0.f, 0.f); }
      sY[r][tx] = make_float4(wA * dA.x, wE * dE.x, wA * dA.y, wE * dE.y);
      sW[r][tx] = make_float2(wA, wE);
    }
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const int k = k0 + r, m = m0 + tx;
    if (m < Nt && k < Nf) {
      const long long o = (long long)k * Nt + m;
      grid[o] = sY[tx][r];
      wgt[o] = sW[tx][r];
    }
  }
}

// ------------------------------------------------------------------------------------------
// Weight structure (a0, C11).  If W[alpha,m,k] = a_alpha[m] b_alpha[k] then
//   rowmax[m] = max_k W = a[m] max b,  colmax[k] = max_m W = b[k] max a,  gmax = max a max b,
// so a'[m] = rowmax[m], b'[k] = colmax[k] / gmax reproduce W = a' b'.  weight_check_kernel counts the
// pixels where that fails by more than a few ulps (or W < 0), and the columns with b' != 1.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
weight_colmax_kernel(const float2* __restrict__ wgt, int Nt, float2* __restrict__ colmax) {   // one block per k
  __shared__ float2 sh[256];
  const int k = blockIdx.x;
  float2 mx = make_float2(0.f, 0.f);
  for (int m = threadIdx.x; m < Nt; m += 256) {
    const float2 w = wgt[(size_t)k * Nt + m];
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

// wa must be zeroed first; grid (ceil(Nt/128), k-slices): weights are >= 0 (or zeroed at upload), so their
// bit patterns order like integers and atomicMax on them is the float maximum
__global__ void weight_rowmax_kernel(const float2* __restrict__ wgt, int Nt, int Nf, float2* __restrict__ wa) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= Nt) return;
  const int per = (Nf + gridDim.y - 1) / gridDim.y;
  const int k0 = blockIdx.y * per, k1 = min(k0 + per, Nf);
  float2 mx = make_float2(0.f, 0.f);
  for (int k = k0; k < k1; ++k) {
    const float2 w = wgt[(size_t)k * Nt + m];
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
                                    const float2* __restrict__ wb, int Nt, int Nf, unsigned long long* counts) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = false;
  if (i < (size_t)Nt * Nf) {
    const int k = (int)(i / Nt), m = (int)(i - (size_t)k * Nt);
    const float2 w = wgt[i], a = wa[m], b = wb[k];
    const float pA = a.x * b.x, pE = a.y * b.y;
    bad = !(fabsf(w.x - pA) <= 1e-6f * pA) || !(fabsf(w.y - pE) <= 1e-6f * pE) || w.x < 0.f || w.y < 0.f;
  }
  const unsigned n_bad = __popc(__ballot_sync(0xffffffffu, bad));
  if ((threadIdx.x & 31) == 0 && n_bad) atomicAdd(&counts[0], (unsigned long long)n_bad);
}

// Compacted list of valid (non-gap) tranches and its prefix counts (C10).  One block.
__global__ void __launch_bounds__(1024)
valid_list_kernel(const uint8_t* __restrict__ gap, int Nt, int* __restrict__ vprefix, int* __restrict__ valid_m) {
  __shared__ int s_cnt[1024];
  const int t = threadIdx.x;
  const int per = (Nt + 1023) / 1024;
  const int b = min(t * per, Nt), e = min(b + per, Nt);
  int c = 0;
  for (int m = b; m < e; ++m) c += gap[m] != 0;
  s_cnt[t] = c;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {                           // inclusive Hillis-Steele scan
    const int v = t >= o ? s_cnt[t - o] : 0;
    __syncthreads();
    s_cnt[t] += v;
    __syncthreads();
  }
  int pos = s_cnt[t] - c;
  for (int m = b; m < e; ++m) {
    vprefix[m] = pos;
    if (gap[m] != 0) valid_m[pos++] = m;
  }
  if (t == 1023) {
    vprefix[Nt] = s_cnt[1023];
    if (s_cnt[1023] == 0) valid_m[0] = 0;                        // keep entry 0 readable when everything is masked
  }
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

__global__ void topk_emit_kernel(const unsigned long long* __restrict__ keys, const float* __restrict__ v,
                                 int k, long long* __restrict__ idx, float* __restrict__ val) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= k) return;
  const unsigned id = 0xFFFFFFFFu - (unsigned)(keys[i] & 0xFFFFFFFFull);
  idx[i] = (long long)id;
  val[i] = v[id];
}

}  // namespace tfs
