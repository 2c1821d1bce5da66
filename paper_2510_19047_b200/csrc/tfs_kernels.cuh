// tfs_kernels.cuh -- device code of libtfs (sm_100a).  See include/tfs.h for the operation and
// DESIGN.md section 6 for the kernel design.  Citations: P:<line> of PAPER.md, C<n> = DESIGN.md.
//
// Work decomposition: one WARP evaluates one (template, time tile) pair.  A time tile is a run
// of <= kTileMax consecutive tranches inside one segment; work items are ordered tile-major so
// that all templates sweep the same slab of the grid together and the slab stays L2-resident.
// Inside a tile lanes are tranches (32 at a time): fp64 0PN track per lane, then each lane walks
// its own window; the grid is stored time-contiguous so those loads coalesce across lanes.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tfs {

#ifndef TFS_WARPS_PER_CTA
#define TFS_WARPS_PER_CTA 24
#endif
constexpr int kWarpsPerCta = TFS_WARPS_PER_CTA;   // one persistent CTA per SM
constexpr int kTileMax = 256;       // tranches per time tile (upper bound)
constexpr int kLutN = 512;          // LUT intervals in t = 1/(1+v)
constexpr double kMtsun = 4.925490947e-6;   // G Msun / c^3 [s]
constexpr double kPi = 3.14159265358979323846;

struct EvalArgs {
  const float4* __restrict__ grid;     // [Nf][Nt] (time-contiguous) {Y_A.re, Y_A.im, Y_E.re, Y_E.im}, Y = W*D
  const float2* __restrict__ wgt;      // [Nf][Nt] {W_A, W_E}
  const uint8_t* __restrict__ gap;     // [Nt] 1 = valid
  const int* __restrict__ vprefix;     // [Nt+1] number of valid tranches before m
  const int* __restrict__ valid_m;     // [vprefix[Nt]] the valid tranche indices, ascending (padded to >= 1 entry)
  const int2* __restrict__ tile_table; // [n_tiles] {i0, i1}: entries of valid_m covered by each tile
  const float4* __restrict__ lut;      // [kLutN+1] {a_F, b_F, a_G, b_G} (see fresnel_aux)
  const double* __restrict__ params;   // [n][8]
  float4* __restrict__ partials;       // [n_tiles][n] {z.re, z.im, hh, 0}
  unsigned long long* bad_count;       // templates rejected (counted on tile 0 only)
  unsigned long long* work_counter;    // next unclaimed work item (zeroed before each launch)
  long long n;                         // templates in this launch
  int Nt, Nf;
  int N_seg, tiles_per_seg, n_tiles;
  int H, adaptive;
  double DT;
  double x_lo, x_hi;                   // band in bins: f_lo*DT, f_hi*DT
  double c_max;
};

// ----- tile geometry: segment n = tranches [ceil(n Nt/N_seg), ceil((n+1) Nt/N_seg))  (C9) -----
__device__ __forceinline__ void tile_range(int tile, int tps, int Nt, int N_seg, int& m0, int& m1) {
  const int n = tile / tps, t = tile - n * tps;
  const int s0 = (int)(((long long)n * Nt + N_seg - 1) / N_seg);
  const int s1 = (int)(((long long)(n + 1) * Nt + N_seg - 1) / N_seg);
  const int L = (s1 - s0 + tps - 1) / tps;
  m0 = min(s0 + t * L, s1);
  m1 = min(m0 + L, s1);
}

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
//   entry i = {a_F, b_F, a_G, b_G}: for t within half a step of i/kLutN,
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

// Returns F = f(|v|)/t, G = g(|v|)/t and ts = sign(v) t, so that sign(v) f = ts F, sign(v) g = ts G.
// lut_lane = shared address of this lane's LUT copy minus kMagicBits * (16 * kLutCopies)  (mod 2^32).
template <int MODE>
__device__ __forceinline__ void fresnel_aux(float v, unsigned lut_lane, float& F, float& G, float& ts) {
  const float a = fabsf(v);
  if (MODE == 0) {
    const float t = rcp_approx(1.0f + a);         // MUFU.RCP
    const float q = fmaf(t, (float)kLutN, kMagic);
    const float4 e = lds128(__float_as_uint(q) * (16u * kLutCopies) + lut_lane);
    ts = copysignf(t, v);
    F = fmaf(t, e.y, e.x);
    G = fmaf(t, e.w, e.z);
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
    F = f;
    G = g;
  }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// dynamic shared memory of kernel A: [LUT copies][fp64 tile sums: 6 per thread, stored [6][threads]]
constexpr int kLutSmemBytes = (kLutN + 1) * kLutCopies * (int)sizeof(float4);
constexpr int kEvalSmemBytes = kLutSmemBytes + 6 * kWarpsPerCta * 32 * (int)sizeof(double);

// One pixel of one tranche (a3-a5).  The template coefficient is h = P h', P = A/sqrt(2c) exp(i phi_m)
// constant over the tranche, and (auxiliary-function form of Eq. 16)
//   h' = s0 G(|v0|) - s1 G(|v1|) E  [+ (1+i) exp(-i pi u^2/c) inside the swept band],  G = g + i f,
//   E = exp(i psi), psi = pi c + 2 pi frac(x).
// The loop accumulates z'_alpha += conj(Y_alpha) h', q'_alpha += W_alpha |h'|^2 and the factor P
// (|P|^2 for q) is applied once per tranche.
struct LaneTrack {      // per-lane (= per-tranche) constants of the pixel loop
  float sc;             // sqrt(2/c)
  float scc;            // sqrt(2c) = v1 - v0
  float hc;             // 1/(2c): pi u^2/c = 2 pi (u^2 hc)
  float Er, Ei;         // exp(i psi)
};

struct LaneSums { float zAr, zAi, zEr, zEi, qA, qE; };

// INBAND: 0 = the pixel is known to lie outside the swept band, 1 = test it (v0 < 0 < v1)
template <int MODE, int INBAND>
__device__ __forceinline__ void pixel(const LaneTrack& L, float u, const float4 Y, const float2 Wt,
                                      unsigned lut_lane, LaneSums& s) {
  const float v0 = L.sc * u;
  const float v1 = v0 + L.scc;
  float F0, G0, t0, F1, G1, t1;
  fresnel_aux<MODE>(v0, lut_lane, F0, G0, t0);
  fresnel_aux<MODE>(v1, lut_lane, F1, G1, t1);
  const float w1r = G1 * L.Er - F1 * L.Ei, w1i = G1 * L.Ei + F1 * L.Er;
  float hr = fmaf(t0, G0, -t1 * w1r);
  float hi = fmaf(t0, F0, -t1 * w1i);
  if (INBAND && v0 < 0.0f && v1 > 0.0f) {
    // pixel inside the swept band: + (1+i) exp(-i pi u^2/c)
    float turns = u * u * L.hc;
    turns -= floorf(turns);
    float st, ct;
    __sincosf(6.283185307179586f * (turns - 0.5f), &st, &ct);        // = -(sin, cos)(2 pi turns)
    hr -= ct + st;
    hi -= ct - st;
  }
  s.zAr = fmaf(Y.x, hr, fmaf(Y.y, hi, s.zAr));
  s.zAi = fmaf(Y.x, hi, fmaf(-Y.y, hr, s.zAi));
  s.zEr = fmaf(Y.z, hr, fmaf(Y.w, hi, s.zEr));
  s.zEi = fmaf(Y.z, hi, fmaf(-Y.w, hr, s.zEi));
  const float h2 = fmaf(hr, hr, hi * hi);
  s.qA = fmaf(Wt.x, h2, s.qA);
  s.qE = fmaf(Wt.y, h2, s.qE);
}

// Generic pixel loop over window offsets [j0, j1): every lane tests its own window length Wm and the
// in-band condition per pixel (wide or clipped windows, ragged tails).  The gather of pixel j+1 is
// issued before the arithmetic of pixel j; lanes past their window run on zeroed data.
template <int MODE>
__device__ __forceinline__ void pixel_loop_generic(const EvalArgs& a, const LaneTrack& L, int j0, int j1, int Wm,
                                                   int idx, float u, unsigned lut_lane, LaneSums& s) {
  float4 Ya = make_float4(0.f, 0.f, 0.f, 0.f), Yb;
  float2 Wa = make_float2(0.f, 0.f), Wb;
  if (j0 < Wm) { Ya = __ldg(a.grid + idx); Wa = __ldg(a.wgt + idx); }
  for (int j = j0; j < j1; j += 2) {
    Yb = make_float4(0.f, 0.f, 0.f, 0.f); Wb = make_float2(0.f, 0.f);
    idx += a.Nt;
    if (j + 1 < Wm) { Yb = __ldg(a.grid + idx); Wb = __ldg(a.wgt + idx); }
    pixel<MODE, 1>(L, u, Ya, Wa, lut_lane, s);
    u -= 1.0f;
    Ya = make_float4(0.f, 0.f, 0.f, 0.f); Wa = make_float2(0.f, 0.f);
    idx += a.Nt;
    if (j + 2 < Wm) { Ya = __ldg(a.grid + idx); Wa = __ldg(a.wgt + idx); }
    pixel<MODE, 1>(L, u, Yb, Wb, lut_lane, s);
    u -= 1.0f;
  }
}

// Fast pixel loop over offsets [0, Wn), Wn <= every active lane's window length: no per-pixel window
// test (inactive lanes never load and keep zeroed data), and the only pixel that can lie inside the
// swept band when c < 1 -- k = ceil(x), offset jc, the same for all lanes -- is singled out by a
// warp-uniform branch.  Loads run two pixels ahead of the arithmetic.
template <int MODE>
__device__ __forceinline__ void pixel_loop_fast(const EvalArgs& a, const LaneTrack& L, int Wn, int jc, bool act,
                                                int idx, float u, unsigned lut_lane, LaneSums& s) {
  float4 Y0 = make_float4(0.f, 0.f, 0.f, 0.f), Y1 = Y0;
  float2 W0 = make_float2(0.f, 0.f), W1 = W0;
  const int Nt = a.Nt;
  if (act) {
    Y0 = __ldg(a.grid + idx); W0 = __ldg(a.wgt + idx);
    if (1 < Wn) { Y1 = __ldg(a.grid + idx + Nt); W1 = __ldg(a.wgt + idx + Nt); }
  }
  // each buffer is refilled (pixel j+2) right after the pixel that used it
  int j = 0;
  for (; j + 2 <= Wn; j += 2) {
    idx += 2 * Nt;
    if (j == jc) pixel<MODE, 1>(L, u, Y0, W0, lut_lane, s); else pixel<MODE, 0>(L, u, Y0, W0, lut_lane, s);
    u -= 1.0f;
    if (act && j + 2 < Wn) { Y0 = __ldg(a.grid + idx); W0 = __ldg(a.wgt + idx); }
    if (j + 1 == jc) pixel<MODE, 1>(L, u, Y1, W1, lut_lane, s); else pixel<MODE, 0>(L, u, Y1, W1, lut_lane, s);
    u -= 1.0f;
    if (act && j + 3 < Wn) { Y1 = __ldg(a.grid + idx + Nt); W1 = __ldg(a.wgt + idx + Nt); }
  }
  if (j < Wn) {
    if (j == jc) pixel<MODE, 1>(L, u, Y0, W0, lut_lane, s); else pixel<MODE, 0>(L, u, Y0, W0, lut_lane, s);
  }
}

// ------------------------------------------------------------------------------------------
// Kernel A: track + gather + per-tile sums.  Persistent: one CTA per SM, warps claim work items
// (template, tile) in tile-major order from a global counter, kClaim at a time.
// Inside a work item LANES ARE TRANCHES: lane l owns the l-th valid (non-gap) tranche of the
// current chunk of 32, computes its track point in fp64 and then walks its own window pixel by
// pixel.  The grid is stored time-contiguous ([k][m]), so the 32 lanes' loads of pixel offset j
// fall on consecutive addresses wherever neighbouring tranches share k_lo (slow chirps: runs of
// 1/c tranches).  Chunks whose active lanes all sweep less than one bin (c < 1: the bulk of every
// bank) and agree on the offset of bin ceil(x) take pixel_loop_fast up to the shortest window and
// finish ragged tails in pixel_loop_generic; all other chunks run pixel_loop_generic throughout.
// ------------------------------------------------------------------------------------------
constexpr int kClaim = 4;

// {i0, i1} = range of the compacted valid-tranche list covered by each tile (C9, C10)
__global__ void tile_table_kernel(const int* __restrict__ vprefix, int Nt, int N_seg, int tps, int n_tiles,
                                  int2* __restrict__ table) {
  const int tile = blockIdx.x * blockDim.x + threadIdx.x;
  if (tile >= n_tiles) return;
  int m0, m1;
  tile_range(tile, tps, Nt, N_seg, m0, m1);
  table[tile] = make_int2(vprefix[m0], vprefix[m1]);
}

template <int MODE>
__global__ void __launch_bounds__(kWarpsPerCta * 32, 1)
eval_tiles_kernel(const EvalArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* s_lut = reinterpret_cast<float4*>(smem_raw);
  double* s_acc = reinterpret_cast<double*>(smem_raw + kLutSmemBytes) + threadIdx.x;   // [6][blockDim]
  constexpr int kAccStride = kWarpsPerCta * 32;

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
      // valid (non-gap) tranches of the tile: entries [i0, i1) of the compacted list (C10)
      const int2 ir = a.tile_table[tile];
      const int i0 = ir.x, i1 = ir.y;

      const TemplateConst T = load_template(a.params + it * 8, a.DT);
      if (!T.ok) {
        if (lane == 0) {
          a.partials[(long long)tile * a.n + it] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (tile == 0) atomicAdd(a.bad_count, 1ULL);
        }
        continue;
      }

      // fp64 per-lane running sums over the tile (z_A, z_E complex, q_A, q_E) live in shared memory
#pragma unroll
      for (int v = 0; v < 6; ++v) s_acc[v * kAccStride] = 0.0;

      for (int ic = i0; ic < i1; ic += 32) {
        // ---------------- track point of this lane's tranche (a2) ----------------
        const int i = ic + lane;
        const bool valid = i < i1;
        const int m = a.valid_m[valid ? i : i0];
        const TrackPoint tp = track_point(T, m, a.DT, a.x_lo, a.x_hi, a.c_max, valid);
        const unsigned act_mask = __ballot_sync(0xffffffffu, tp.active);
        if (act_mask == 0u) continue;
        int Wm = 0, idx = 0, jc = -1;
        float u = 0.f, Pr = 0.f, Pi = 0.f;
        LaneTrack L;
        L.sc = 1.f; L.scc = 1.f; L.hc = 0.f; L.Er = 0.f; L.Ei = 0.f;
        if (tp.active) {
          int k_lo, k_hi;
          window(tp, a.H, a.adaptive, a.Nf, k_lo, k_hi);
          Wm = k_hi - k_lo + 1;
          idx = k_lo * a.Nt + m;
          const double flx = floor(tp.x);
          const float fracx = (float)(tp.x - flx);
          u = fracx - (float)(k_lo - (int)flx);          // cancellation-safe x - k_lo
          jc = (int)ceil(tp.x) - k_lo;                   // offset of bin ceil(x)
          // phases in turns, reduced in fp64 (phi reaches ~1e8 rad), then to [-1/2, 1/2)
          double tphi = T.phic_turns - tp.X58 * (1.0 / kPi);
          tphi -= floor(tphi);
          double tpsi = 0.5 * tp.c + (tp.x - flx);
          tpsi -= floor(tpsi);
          float sphi, cphi, spsi, cpsi;
          __sincosf(6.283185307179586f * ((float)tphi - 0.5f), &sphi, &cphi);     // = -(sin, cos)(2 pi tphi)
          __sincosf(6.283185307179586f * ((float)tpsi - 0.5f), &spsi, &cpsi);
          const float cf = (float)tp.c;
          const float pre = -(T.acoef * tp.Xm14) * rsqrtf(2.0f * cf);           // -A_m / sqrt(2c)
          L.sc = rsqrtf(0.5f * cf);
          L.scc = L.sc * cf;
          L.hc = __fdividef(0.5f, cf);
          Pr = pre * cphi;
          Pi = pre * sphi;
          L.Er = -cpsi;
          L.Ei = -spsi;
        }
        // warp-uniform choice of the pixel loop
        const int Wmax = __reduce_max_sync(0xffffffffu, Wm);
        const int Wmin = __reduce_min_sync(0xffffffffu, tp.active ? Wm : 0x7fffffff);
        const int jc0 = __shfl_sync(0xffffffffu, jc, __ffs(act_mask) - 1);
        const bool fast_lane = !tp.active || (tp.c < 1.0 && jc == jc0);
        const bool fast = __all_sync(0xffffffffu, fast_lane) && jc0 >= 0 && jc0 < Wmin;

        // ---------------- pixel loop (a3-a5): lane walks its own window ----------------
        LaneSums s;
        s.zAr = 0.f; s.zAi = 0.f; s.zEr = 0.f; s.zEi = 0.f; s.qA = 0.f; s.qE = 0.f;
        if (fast) {
          pixel_loop_fast<MODE>(a, L, Wmin, jc0, tp.active, idx, u, lut_lane, s);
          if (Wmax > Wmin)
            pixel_loop_generic<MODE>(a, L, Wmin, Wmax, Wm, idx + Wmin * a.Nt, u - (float)Wmin, lut_lane, s);
        } else {
          pixel_loop_generic<MODE>(a, L, 0, Wmax, Wm, idx, u, lut_lane, s);
        }
        // apply the tranche's factor P (and |P|^2) and promote to fp64
        const float P2 = fmaf(Pr, Pr, Pi * Pi);
        s_acc[0 * kAccStride] += (double)(Pr * s.zAr - Pi * s.zAi);
        s_acc[1 * kAccStride] += (double)(Pr * s.zAi + Pi * s.zAr);
        s_acc[2 * kAccStride] += (double)(Pr * s.zEr - Pi * s.zEi);
        s_acc[3 * kAccStride] += (double)(Pr * s.zEi + Pi * s.zEr);
        s_acc[4 * kAccStride] += (double)(P2 * s.qA);
        s_acc[5 * kAccStride] += (double)(P2 * s.qE);
      }

      const double dzAr = warp_sum(s_acc[0 * kAccStride]), dzAi = warp_sum(s_acc[1 * kAccStride]);
      const double dzEr = warp_sum(s_acc[2 * kAccStride]), dzEi = warp_sum(s_acc[3 * kAccStride]);
      const double dqA = warp_sum(s_acc[4 * kAccStride]),  dqE = warp_sum(s_acc[5 * kAccStride]);
      if (lane == 0) {
        // z = T_A z_A + T_E z_E ; hh = |T_A|^2 q_A + |T_E|^2 q_E   (Eq. 29, Eq. 31)
        const double zr = T.TAr * dzAr - T.TAi * dzAi + T.TEr * dzEr - T.TEi * dzEi;
        const double zi = T.TAr * dzAi + T.TAi * dzAr + T.TEr * dzEi + T.TEi * dzEr;
        const double hh = (T.TAr * T.TAr + T.TAi * T.TAi) * dqA + (T.TEr * T.TEr + T.TEi * T.TEi) * dqE;
        a.partials[(long long)tile * a.n + it] = make_float4((float)zr, (float)zi, (float)hh, 0.f);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// Kernel B: sum tile partials per segment, P_n = |z_n|^2/hh_n, Upsilon = sum_n P_n (Eq. 8, 9).
// ------------------------------------------------------------------------------------------
__global__ void combine_kernel(const float4* __restrict__ partials, long long n, int N_seg, int tps,
                               float* __restrict__ upsilon, float* __restrict__ seg_power,
                               float* __restrict__ seg_dh, float* __restrict__ seg_hh) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double ups = 0.0;
  for (int s = 0; s < N_seg; ++s) {
    double zr = 0, zi = 0, hh = 0;
    for (int t = 0; t < tps; ++t) {
      const float4 p = partials[(long long)(s * tps + t) * n + i];
      zr += p.x; zi += p.y; hh += p.z;
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
      const float2 dA = coeff[i], dE = coeff[npix + i];
      const float wA = weight ? weight[i] : 1.0f;
      const float wE = weight ? weight[npix + i] : 1.0f;
      sY[r][tx] = make_float4(wA * dA.x, wA * dA.y, wE * dE.x, wE * dE.y);
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

__global__ void topk_emit_kernel(const unsigned long long* __restrict__ keys, const float* __restrict__ v,
                                 int k, long long* __restrict__ idx, float* __restrict__ val) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= k) return;
  const unsigned id = 0xFFFFFFFFu - (unsigned)(keys[i] & 0xFFFFFFFFull);
  idx[i] = (long long)id;
  val[i] = v[id];
}

}  // namespace tfs
