// tfs_kernels.cuh -- device code of libtfs (sm_100a).  See include/tfs.h for the operation and
// DESIGN.md section 6 for the kernel design.  Citations: P:<line> of PAPER.md, C<n> = DESIGN.md.
//
// Work decomposition: one WARP evaluates one (template, time tile) pair.  A time tile is a run
// of <= TILE_MAX consecutive tranches inside one segment; work items are ordered tile-major so
// that all templates sweep the same slab of the grid together and the slab stays L2-resident.
// Inside a tile the warp alternates, per chunk of 32 tranches, between
//   phase 1: lane <-> tranche: fp64 0PN track, window, phases  -> per-tranche record in smem
//   phase 2: lane <-> (tranche, pixel) item of the flattened window list: Fresnel-kernel value
//            from the auxiliary-function LUT, 16-byte gather of both channels, accumulate.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tfs {

constexpr int kWarpsPerCta = 32;       // one 1024-thread CTA per SM
constexpr int kChunk = 32;          // tranches per phase-1 pass (one per lane)
constexpr int kLutN = 512;          // LUT intervals in t = 1/(1+v)
constexpr double kMtsun = 4.925490947e-6;   // G Msun / c^3 [s]
constexpr double kPi = 3.14159265358979323846;

struct EvalArgs {
  const float4* __restrict__ grid;     // [Nt][Nf] {Y_A.re, Y_A.im, Y_E.re, Y_E.im}, Y = W*D
  const float2* __restrict__ wgt;      // [Nt][Nf] {W_A, W_E}
  const uint8_t* __restrict__ gap;     // [Nt] 1 = valid
  const float4* __restrict__ lut;      // [kLutN+1] {F, F', G, G'} (see fresnel_aux)
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

// Per-tranche record consumed by phase 2 (48 bytes, in shared memory).
struct __align__(16) BinRec {
  int base;      // m*Nf + k_lo
  int W;         // window width
  float u0;      // x - k_lo
  float sc;      // sqrt(2/c)
  float Pr, Pi;  // A/sqrt(2c) * exp(i phi_m)
  float Qr, Qi;  // P * exp(i psi), psi = pi c + 2 pi frac(x)
  float scc;     // sqrt(2/c)*c = sqrt(2c)
  float hc;      // 1/(2c): pi u^2/c = 2 pi * (u^2 * hc)
  float pad0, pad1;
};

// LUT of the Fresnel auxiliary functions, indexed by round(t*kLutN), t = 1/(1+|v|):
//   entry i = {F_i, F'_i, G_i, G'_i},  f(v) = t (F_i + fr F'_i),  g(v) = t (G_i + fr G'_i),  fr = t*kLutN - i
// (F = f/t, G = g/t, primes = central differences per index step).  In shared memory it is stored
// kLutCopies times, copy r at 16-byte slot (i*kLutCopies + r), and lane l reads copy l & 7: the 8
// lanes of a quarter-warp then always hit 8 different bank groups, so an LDS.128 is conflict-free
// whatever the indices are (measured 9 wavefronts per load without the copies, 4 with).
constexpr int kLutCopies = 8;
constexpr float kMagic = 12582912.0f;          // 1.5 * 2^23: (p + kMagic) rounds p to an integer in the mantissa

template <int MODE>
__device__ __forceinline__ void fresnel_aux(float v, const float4* __restrict__ lut_lane, float& f, float& g) {
  // Returns sign(v) f(|v|), sign(v) g(|v|).
  // MODE 0: LUT;  MODE 1: the paper's Eqs. 27-28 (|v| <= 6) and the plain asymptote
  // f = 1/(pi v), g = 0 (Eqs. 23-24, |v| > 6).
  const float a = fabsf(v);
  if (MODE == 0) {
    const float t = __fdividef(1.0f, 1.0f + a);
    const float q = fmaf(t, (float)kLutN, kMagic);
    const float fr = fmaf(t, (float)kLutN, -(q - kMagic));
    const int i = __float_as_int(q) - __float_as_int(kMagic);
    const float4 e = lut_lane[i * kLutCopies];
    const float ts = copysignf(t, v);
    f = ts * fmaf(fr, e.y, e.x);
    g = ts * fmaf(fr, e.w, e.z);
  } else {
    if (a > 6.0f) {
      f = __fdividef(0.318309886183790672f, a);
      g = 0.0f;
    } else {
      f = __fdividef(1.0f + 0.926f * a, 2.0f + a * (1.792f + 3.104f * a));
      g = __fdividef(1.0f, 2.0f + a * (4.142f + a * (3.492f + 6.670f * a)));
    }
    f = copysignf(f, v);
    g = copysignf(g, v);
  }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// dynamic shared memory of kernel A: [LUT copies][records of every warp]
constexpr int kLutSmemBytes = (kLutN + 1) * kLutCopies * (int)sizeof(float4);
constexpr int kEvalSmemBytes = kLutSmemBytes + kWarpsPerCta * kChunk * (int)sizeof(BinRec);

// ------------------------------------------------------------------------------------------
// Kernel A: track + gather + per-tile sums.  Persistent: one CTA per SM, warps claim work items
// (template, tile) in tile-major order from a global counter, kClaim at a time.
// ------------------------------------------------------------------------------------------
constexpr int kClaim = 4;

template <int MODE>
__global__ void __launch_bounds__(kWarpsPerCta * 32, 1)
eval_tiles_kernel(const EvalArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* s_lut = reinterpret_cast<float4*>(smem_raw);
  BinRec* s_rec = reinterpret_cast<BinRec*>(smem_raw + kLutSmemBytes);

  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  if (MODE == 0) {
    for (int i = threadIdx.x; i < (kLutN + 1) * kLutCopies; i += blockDim.x) s_lut[i] = a.lut[i / kLutCopies];
    __syncthreads();
  }
  BinRec* rec = s_rec + warp * kChunk;
  const float4* lut_lane = s_lut + (lane & (kLutCopies - 1));

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

      const TemplateConst T = load_template(a.params + it * 8);
      if (!T.ok) {
        if (lane == 0) {
          a.partials[(long long)tile * a.n + it] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (tile == 0) atomicAdd(a.bad_count, 1ULL);
        }
        continue;
      }

      // fp64 per-lane running sums over the tile: z_A, z_E (complex), q_A, q_E
      double dzAr = 0, dzAi = 0, dzEr = 0, dzEi = 0, dqA = 0, dqE = 0;

      for (int mc = m0; mc < m1; mc += kChunk) {
        // ---------------- phase 1: lane <-> tranche ----------------
        const int m = mc + lane;
        const bool valid = (m < m1) && (a.gap[min(m, a.Nt - 1)] != 0);        // C10
        const TrackPoint tp = track_point(T, m, a.DT, a.x_lo, a.x_hi, a.c_max, valid);
        const unsigned act_mask = __ballot_sync(0xffffffffu, tp.active);
        if (act_mask == 0u) continue;
        int Wm = 0;
        if (tp.active) {
          int k_lo, k_hi;
          window(tp, a.H, a.adaptive, a.Nf, k_lo, k_hi);
          Wm = k_hi - k_lo + 1;
          const double flx = floor(tp.x);
          const float fracx = (float)(tp.x - flx);
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
          BinRec r;
          r.base = m * a.Nf + k_lo;
          r.W = Wm;
          r.u0 = fracx - (float)(k_lo - (int)flx);      // cancellation-safe x - k_lo
          r.sc = rsqrtf(0.5f * cf);
          r.Pr = pre * cphi;
          r.Pi = pre * sphi;
          r.Qr = r.Pr * cpsi - r.Pi * spsi;
          r.Qi = r.Pr * spsi + r.Pi * cpsi;
          r.scc = r.sc * cf;
          r.hc = __fdividef(0.5f, cf);
          r.pad0 = 0.f; r.pad1 = 0.f;
          const int slot = __popc(act_mask & ((1u << lane) - 1u));
          rec[slot] = r;
        }
        int Wc = Wm;                                                          // chunk-uniform width
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) Wc = max(Wc, __shfl_xor_sync(0xffffffffu, Wc, o));
        __syncwarp();

        // ---------------- phase 2: lane <-> (tranche, pixel) item ----------------
        // item i -> (slot b, offset j) = (i / Wc, i % Wc), advanced incrementally; the gather of
        // item i+32 is issued before the arithmetic of item i (software prefetch, distance 1).
        const int n_items = __popc(act_mask) * Wc;
        float zAr = 0, zAi = 0, zEr = 0, zEi = 0, qA = 0, qE = 0;
        int b = 0, j = lane;
        while (j >= Wc) { j -= Wc; ++b; }
        float4 Yn = make_float4(0.f, 0.f, 0.f, 0.f);
        float2 Wn = make_float2(0.f, 0.f);
        float un = 0.f, scn = 0.f;
        bool vn = false;
        if (lane < n_items) {
          const float4 h = *reinterpret_cast<const float4*>(&rec[b]);          // {base, W, u0, sc}
          vn = j < __float_as_int(h.y);
          if (vn) {
            const int idx = __float_as_int(h.x) + j;
            Yn = __ldg(a.grid + idx);
            Wn = __ldg(a.wgt + idx);
            un = h.z - (float)j;
            scn = h.w;
          }
        }
        for (int i = lane; i < n_items; i += 32) {
          const float4 Y = Yn;
          const float2 Wt = Wn;
          const float u = un, sc = scn;
          const bool vc = vn;
          const BinRec* rc = rec + b;
          // ---- prefetch item i+32 ----
          j += 32;
          while (j >= Wc) { j -= Wc; ++b; }
          vn = false;
          if (i + 32 < n_items) {
            const float4 h = *reinterpret_cast<const float4*>(&rec[b]);
            vn = j < __float_as_int(h.y);
            if (vn) {
              const int idx = __float_as_int(h.x) + j;
              Yn = __ldg(a.grid + idx);
              Wn = __ldg(a.wgt + idx);
              un = h.z - (float)j;
              scn = h.w;
            }
          }
          // ---- arithmetic of item i ----
          if (vc) {
            const float4 PQ = *reinterpret_cast<const float4*>(&rc->Pr);       // {Pr, Pi, Qr, Qi}
            const float scc = rc->scc;
            const float v0 = sc * u;
            const float v1 = v0 + scc;
            float f0, g0, f1, g1;
            fresnel_aux<MODE>(v0, lut_lane, f0, g0);
            fresnel_aux<MODE>(v1, lut_lane, f1, g1);
            // s0 G(|v0|) P - s1 G(|v1|) Q,  G = g + i f   (C7)
            float hr = g0 * PQ.x - f0 * PQ.y - g1 * PQ.z + f1 * PQ.w;
            float hi = g0 * PQ.y + f0 * PQ.x - g1 * PQ.w - f1 * PQ.z;
            if (v0 < 0.0f && v1 > 0.0f) {
              // pixel inside the swept band: + (1+i) exp(-i pi u^2/c) P
              float turns = u * u * rc->hc;
              turns -= floorf(turns);
              float st, ct;
              __sincosf(6.283185307179586f * (turns - 0.5f), &st, &ct);        // = -(sin, cos)(2 pi turns)
              const float er = -(ct + st), ei = -(ct - st);
              hr += er * PQ.x - ei * PQ.y;
              hi += er * PQ.y + ei * PQ.x;
            }
            zAr = fmaf(Y.x, hr, fmaf(Y.y, hi, zAr));
            zAi = fmaf(Y.x, hi, fmaf(-Y.y, hr, zAi));
            zEr = fmaf(Y.z, hr, fmaf(Y.w, hi, zEr));
            zEi = fmaf(Y.z, hi, fmaf(-Y.w, hr, zEi));
            const float h2 = fmaf(hr, hr, hi * hi);
            qA = fmaf(Wt.x, h2, qA);
            qE = fmaf(Wt.y, h2, qE);
          }
        }
        dzAr += zAr; dzAi += zAi; dzEr += zEr; dzEi += zEi; dqA += qA; dqE += qE;
        __syncwarp();
      }

      dzAr = warp_sum(dzAr); dzAi = warp_sum(dzAi);
      dzEr = warp_sum(dzEr); dzEi = warp_sum(dzEi);
      dqA = warp_sum(dqA);   dqE = warp_sum(dqE);
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
// Upload: Y = W*D interleaved by channel, W interleaved.
// ------------------------------------------------------------------------------------------
__global__ void pack_kernel(const float2* __restrict__ coeff, const float* __restrict__ weight,
                            long long npix, float4* __restrict__ grid, float2* __restrict__ wgt) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npix) return;
  const float2 dA = coeff[i], dE = coeff[npix + i];
  const float wA = weight ? weight[i] : 1.0f;
  const float wE = weight ? weight[npix + i] : 1.0f;
  grid[i] = make_float4(wA * dA.x, wA * dA.y, wE * dE.x, wE * dE.y);
  wgt[i] = make_float2(wA, wE);
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
