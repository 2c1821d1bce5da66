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

// Per-template constants derived from the parameter row (all fp64).
struct TemplateConst {
  double tc, phic_turns, inv5M, xcoef, acoef;
  double TAr, TAi, TEr, TEi;
  bool ok;
};

__device__ __forceinline__ TemplateConst load_template(const double* __restrict__ p) {
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
  t.xcoef = 1.0 / (8.0 * kPi * M);                        // f = X^{-3/8} * xcoef ; x = f*DT
  // A_m = amp f^{2/3} = amp (8 pi M)^{-2/3} X^{-1/4}
  t.acoef = (ok ? amp : 0.0) * cbrt(t.xcoef * t.xcoef);
  t.phic_turns = (ok ? phic : 0.0) * (0.5 / kPi);
  t.ok = ok;
  return t;
}

// Track point of one tranche (Eqs. 12-15 at the tranche start, C6; 0PN, C5).
struct TrackPoint {
  double x;        // f_m * DT  (position in bins)
  double c;        // fdot_m * DT^2 (bins swept in the tranche)
  double X58;      // X^{5/8}: phi_m = phic - 2 X^{5/8}
  double Xm14;     // X^{-1/4}: A_m = acoef * X^{-1/4}
  bool active;
};

__device__ __forceinline__ TrackPoint track_point(const TemplateConst& t, int m, double DT,
                                                  double x_lo, double x_hi, double c_max, bool valid) {
  TrackPoint r;
  const double tau = t.tc - (double)m * DT;
  bool act = valid && (tau > DT);
  const double X = act ? tau * t.inv5M : 1.0;
  // X^{1/2}, X^{1/4}, X^{1/8} by a chain of reciprocal square roots
  const double r1 = rsqrt(X);        // X^{-1/2}
  const double s1 = X * r1;          // X^{ 1/2}
  const double r2 = rsqrt(s1);       // X^{-1/4}
  const double s2 = s1 * r2;         // X^{ 1/4}
  const double r3 = rsqrt(s2);       // X^{-1/8}
  const double s3 = s2 * r3;         // X^{ 1/8}
  r.X58 = s1 * s3;
  r.Xm14 = r2;
  r.x = (s3 * r1) * (t.xcoef * DT);  // X^{-3/8} / (8 pi M) * DT
  r.c = 0.375 * r.x * DT / (act ? tau : 1.0);      // fdot DT^2 = 3 f DT^2 / (8 tau)
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

// One pixel of one tranche (a3-a5): template coefficient from the auxiliary-function form of Eq. 16
// (DESIGN.md section 6.3), then z_alpha += Y_alpha^* h, q_alpha += W_alpha |h|^2 for both channels.
struct LaneTrack {      // per-lane (= per-tranche) constants of the pixel loop
  float sc;             // sqrt(2/c)
  float scc;            // sqrt(2c) = v1 - v0
  float hc;             // 1/(2c): pi u^2/c = 2 pi (u^2 hc)
  float Pr, Pi;         // A/sqrt(2c) exp(i phi_m)
  float Qr, Qi;         // P exp(i psi), psi = pi c + 2 pi frac(x)
};

struct LaneSums { float zAr, zAi, zEr, zEi, qA, qE; };

template <int MODE>
__device__ __forceinline__ void pixel(const LaneTrack& L, float u, const float4 Y, const float2 Wt,
                                      unsigned lut_lane, LaneSums& s) {
  const float v0 = L.sc * u;
  const float v1 = v0 + L.scc;
  float F0, G0, t0, F1, G1, t1;
  fresnel_aux<MODE>(v0, lut_lane, F0, G0, t0);
  fresnel_aux<MODE>(v1, lut_lane, F1, G1, t1);
  // h = s0 G(|v0|) P - s1 G(|v1|) Q,  G = g + i f
  const float w0r = G0 * L.Pr - F0 * L.Pi, w0i = G0 * L.Pi + F0 * L.Pr;
  const float w1r = G1 * L.Qr - F1 * L.Qi, w1i = G1 * L.Qi + F1 * L.Qr;
  float hr = fmaf(t0, w0r, -t1 * w1r);
  float hi = fmaf(t0, w0i, -t1 * w1i);
  if (v0 < 0.0f && v1 > 0.0f) {
    // pixel inside the swept band: + (1+i) exp(-i pi u^2/c) P
    float turns = u * u * L.hc;
    turns -= floorf(turns);
    float st, ct;
    __sincosf(6.283185307179586f * (turns - 0.5f), &st, &ct);        // = -(sin, cos)(2 pi turns)
    const float er = -(ct + st), ei = -(ct - st);
    hr += er * L.Pr - ei * L.Pi;
    hi += er * L.Pi + ei * L.Pr;
  }
  s.zAr = fmaf(Y.x, hr, fmaf(Y.y, hi, s.zAr));
  s.zAi = fmaf(Y.x, hi, fmaf(-Y.y, hr, s.zAi));
  s.zEr = fmaf(Y.z, hr, fmaf(Y.w, hi, s.zEr));
  s.zEi = fmaf(Y.z, hi, fmaf(-Y.w, hr, s.zEi));
  const float h2 = fmaf(hr, hr, hi * hi);
  s.qA = fmaf(Wt.x, h2, s.qA);
  s.qE = fmaf(Wt.y, h2, s.qE);
}

// ------------------------------------------------------------------------------------------
// Kernel A: track + gather + per-tile sums.  Persistent: one CTA per SM, warps claim work items
// (template, tile) in tile-major order from a global counter, kClaim at a time.
// Inside a work item LANES ARE TRANCHES: lane l owns the l-th valid (non-gap) tranche of the
// current chunk of 32, computes its track point in fp64 and then walks its own window pixel by
// pixel.  The grid is stored time-contiguous ([k][m]), so the 32 lanes' loads of pixel offset j
// fall on consecutive addresses wherever neighbouring tranches share k_lo (slow chirps: runs of
// 1/c tranches).  Lanes past their window (or inactive) keep running with zeroed data: the loop has
// no divergent branch except the rare in-band term.
// ------------------------------------------------------------------------------------------
constexpr int kClaim = 4;

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
    const long long w1 = min(w0 + kClaim, n_work);
    for (long long w = w0; w < w1; ++w) {
      const int tile = (int)(w / a.n);
      const long long it = w - (long long)tile * a.n;
      int m0, m1;
      tile_range(tile, a.tiles_per_seg, a.Nt, a.N_seg, m0, m1);
      // valid (non-gap) tranches of the tile: entries [i0, i1) of the compacted list (C10)
      const int i0 = a.vprefix[m0], i1 = a.vprefix[m1];

      const TemplateConst T = load_template(a.params + it * 8);
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
        if (__ballot_sync(0xffffffffu, tp.active) == 0u) continue;
        int Wm = 0, idx = 0;
        float u = 0.f;
        LaneTrack L;
        L.sc = 1.f; L.scc = 1.f; L.hc = 0.f; L.Pr = 0.f; L.Pi = 0.f; L.Qr = 0.f; L.Qi = 0.f;
        if (tp.active) {
          int k_lo, k_hi;
          window(tp, a.H, a.adaptive, a.Nf, k_lo, k_hi);
          Wm = k_hi - k_lo + 1;
          idx = k_lo * a.Nt + m;
          const double flx = floor(tp.x);
          const float fracx = (float)(tp.x - flx);
          u = fracx - (float)(k_lo - (int)flx);          // cancellation-safe x - k_lo
          // phases in turns, reduced in fp64 (phi reaches ~1e8 rad)
          double tphi = T.phic_turns - tp.X58 * (1.0 / kPi);
          tphi -= floor(tphi);
          double tpsi = 0.5 * tp.c + (tp.x - flx);
          tpsi -= floor(tpsi);
          float sphi, cphi, spsi, cpsi;
          sincospif(2.0f * (float)tphi, &sphi, &cphi);
          sincospif(2.0f * (float)tpsi, &spsi, &cpsi);
          const float cf = (float)tp.c;
          const float pre = (float)(T.acoef * tp.Xm14) * rsqrtf(2.0f * cf);  // A_m / sqrt(2c)
          L.sc = rsqrtf(0.5f * cf);
          L.scc = L.sc * cf;
          L.hc = __fdividef(0.5f, cf);
          L.Pr = pre * cphi;
          L.Pi = pre * sphi;
          L.Qr = L.Pr * cpsi - L.Pi * spsi;
          L.Qi = L.Pr * spsi + L.Pi * cpsi;
        }
        const int Wmax = __reduce_max_sync(0xffffffffu, Wm);

        // ---------------- pixel loop (a3-a5): lane walks its own window ----------------
        // the gather of pixel j+1 is issued before the arithmetic of pixel j
        LaneSums s;
        s.zAr = 0.f; s.zAi = 0.f; s.zEr = 0.f; s.zEi = 0.f; s.qA = 0.f; s.qE = 0.f;
        float4 Ya = make_float4(0.f, 0.f, 0.f, 0.f), Yb;
        float2 Wa = make_float2(0.f, 0.f), Wb;
        if (0 < Wm) { Ya = __ldg(a.grid + idx); Wa = __ldg(a.wgt + idx); }
        for (int j = 0; j < Wmax; j += 2) {
          Yb = make_float4(0.f, 0.f, 0.f, 0.f); Wb = make_float2(0.f, 0.f);
          idx += a.Nt;
          if (j + 1 < Wm) { Yb = __ldg(a.grid + idx); Wb = __ldg(a.wgt + idx); }
          pixel<MODE>(L, u, Ya, Wa, lut_lane, s);
          u -= 1.0f;
          Ya = make_float4(0.f, 0.f, 0.f, 0.f); Wa = make_float2(0.f, 0.f);
          idx += a.Nt;
          if (j + 2 < Wm) { Ya = __ldg(a.grid + idx); Wa = __ldg(a.wgt + idx); }
          pixel<MODE>(L, u, Yb, Wb, lut_lane, s);
          u -= 1.0f;
        }
        s_acc[0 * kAccStride] += s.zAr; s_acc[1 * kAccStride] += s.zAi;
        s_acc[2 * kAccStride] += s.zEr; s_acc[3 * kAccStride] += s.zEi;
        s_acc[4 * kAccStride] += s.qA;  s_acc[5 * kAccStride] += s.qE;
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
  const TemplateConst T = load_template(a.params + w * 8);
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
