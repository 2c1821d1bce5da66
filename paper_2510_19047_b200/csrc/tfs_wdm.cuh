// tfs_wdm.cuh -- the statistic on real-coefficient orthonormal WDM wavelet pixels (SURVEY.md 8(f) NEXT-1,
// DESIGN.md section 12; BASELINE.json north_star: "wavelet-pixel" data in an "orthonormal TF basis").
// The paper works on complex short-time Fourier tranches and only cites wavelet methods; the
// basis equations are in its ref. [28], not in the container, so this follows the standard
// Wilson-Daubechies-Meyer construction under the readings W1-W7 of DESIGN.md:
//   grid     Nt time pixels x Nf layers of real coefficients, pixel duration DT = Nf dt, layer spacing DF = 1/(2 DT)
//   window   Phi(omega) = cos(pi |omega| / (2 DOmega)) on |omega| <= DOmega (Meyer condition, no flat top)
//   pixel    H_nm = eps_nm (A_n/sqrt2) exp(i Phi_n) K(x, kappa),  x = f_n/DF - m,  kappa = 4 fdot_n DT^2,
//            track expanded about the pixel CENTRE t_n = n DT (Eqs. 12-15 moved there),
//            eps = 1 (n + m even), i (-1)^(n m) (n + m odd),
//            K = response of the window to a linear chirp, in closed form through the Fresnel integrals:
//              K = exp(i pi/4)/(2 sqrt2) sum_{s=+-1} exp(i pi kappa/16 - s i pi x/2) conj[F(v_hi,s) - F(v_lo,s)],
//              v_{hi,lo;s} = sqrt(2/kappa) (x +- 1 - s kappa/4)
//   stat     per segment [a b] G^-1 [a b]^T, a + i b = sum_alpha sum W d (T_alpha H), G the 2x2 Gram matrix
//            of (Re, Im)(T_alpha H) under W: each segment maximised over amplitude and phase (Eq. 5)
// As for Eq. 16 the Fresnel differences are evaluated without cancellation through the
// auxiliary functions: with Godd(v) = sign(v) (g + i f)(|v|) and the two large phases
// E_hi = exp(-i pi (x+1)^2/kappa), E_lo = exp(-i pi (x-1)^2/kappa) reduced in fp64,
//   K = exp(i pi kappa/16)/2 [in_+ exp(-i pi x/2) + in_- exp(+i pi x/2)]
//       + exp(-i pi/4)/(2 sqrt2) [E_hi conj(Godd(v_hi,+) - Godd(v_hi,-)) + E_lo conj(Godd(v_lo,+) - Godd(v_lo,-))]
// with in_s = 1 when v_lo,s < 0 < v_hi,s.  The auxiliary functions come from the same shared-memory table
// as the near zone of the Fourier path ("the wavelet filter-response lookup table staged in shared memory").
//
// Work decomposition: the list machinery of tfs_kernels.cuh -- items (template, tile of kTS valid time
// pixels) in tile-major order, one warp per item, lanes are time pixels, pieces cut at segment boundaries.
// Data layout: y[m][i] = {W_0 d_0, W_1 d_1}, w[m][i] = {W_0, W_1}, float2, time-contiguous over the valid pixels.
#pragma once
#include "tfs_kernels.cuh"

namespace tfs {

struct Cplx { float r, i; };
__device__ __forceinline__ Cplx cmulf(Cplx a, Cplx b) { return {a.r * b.r - a.i * b.i, a.r * b.i + a.i * b.r}; }

// Godd(v) = sign(v) (g(|v|) + i f(|v|)) from the shared-memory table
__device__ __forceinline__ Cplx godd(float v, unsigned lut_lane) {
  f2_t GF;
  float ts, g, f;
  fresnel_aux<0, kLutCopiesList>(v, lut_lane, GF, ts);
  upk(GF, g, f);
  return {ts * g, ts * f};
}

// One WDM work item: template `it` on time tile `tile`.  Writes, per piece, {a, b, hcc, hss} and {hcs, 0, 0, 0}.
__device__ __forceinline__ void eval_item_wdm(const EvalArgs& a, const long long it, const int tile, const int lane,
                                              const unsigned lut_lane) {
  const TplConst T = a.tconst[it];
  const float2* __restrict__ gy = reinterpret_cast<const float2*>(a.grid);
  const float2* __restrict__ gw = a.wgt;
  const int i0 = tile * kTS, i1 = min(i0 + kTS, a.n_valid);
  int p = a.tile_first[tile];
  const int p_stop = a.tile_first[tile + 1];
  int pend = p < p_stop ? a.piece_end[p] : i1;
  float acc[5] = {0.f, 0.f, 0.f, 0.f, 0.f};

  auto flush = [&]() {
    float r[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) { r[q] = acc[q]; acc[q] = 0.f; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
      for (int q = 0; q < 5; ++q) r[q] += __shfl_xor_sync(0xffffffffu, r[q], o);
    }
    if (lane == 0) {
      float4* dst = a.partials + ((long long)p * a.n + it) * 2;
      dst[0] = make_float4(r[0], r[1], r[2], r[3]);
      dst[1] = make_float4(r[4], 0.f, 0.f, 0.f);
    }
  };

  for (int ic = i0; ic < i1; ic += 32) {
    const int i = ic + lane;
    const bool valid = i < i1;
    const int n_pix = a.valid_m[valid ? i : i0];
    const TrackPoint tp = track_point_at(T, (double)n_pix * a.wdm_DTpix, a.DT, a.x_lo, a.x_hi, a.c_max, 0.5, valid);
    const unsigned act_mask = __ballot_sync(0xffffffffu, tp.active);
    const int cend = min(ic + 32, i1);
    const bool closes = p < p_stop && pend <= cend;
    float v[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
    if (act_mask != 0u) {
      int m_lo = 1, Wm = 0, kfl = 0;
      double fr = 0.0, inv2k = 0.0;
      float sc = 1.f, kq = 0.125f;
      Cplx eK = {1.f, 0.f}, P = {0.f, 0.f};
      if (tp.active) {
        kfl = __double2int_rd(tp.x);
        fr = tp.x - (double)kfl;
        const int kce = fr > 0.0 ? kfl + 1 : kfl;                       // ceil(x)
        m_lo = max(kce - 1 - a.wdm_Hw, 1);
        const int m_hi = min(kfl + 1 + a.wdm_Hw, a.Nf - 1);
        m_lo = min(m_lo, a.Nf - 1);
        Wm = max(m_hi - m_lo + 1, 0);
        const float kf = (float)tp.c;                                   // kappa = 4 fdot DT^2
        inv2k = 0.5 / tp.c;
        sc = rsqrt_approx(0.5f * kf);
        kq = 0.25f * kf;
        float s1, c1;
        __sincosf(0.19634954084936207f * kf, &s1, &c1);                 // pi kappa / 16
        eK = {c1, s1};
        double tphi = T.phic_turns - tp.X58 * (1.0 / kPi);
        tphi -= floor(tphi);
        float sphi, cphi;
        __sincosf(6.283185307179586f * ((float)tphi - 0.5f), &sphi, &cphi);   // = -(sin, cos)(2 pi tphi)
        const float amp = -(T.acoef * tp.Xm14) * 0.70710678118654752f;        // -A_n / sqrt2
        P = {amp * cphi, amp * sphi};
      }
      const int Wmax = __reduce_max_sync(0xffffffffu, Wm);
      Cplx z0 = {0.f, 0.f}, z1 = {0.f, 0.f}, S20 = {0.f, 0.f}, S21 = {0.f, 0.f};
      float S00 = 0.f, S01 = 0.f;
      const int col = valid ? i : i0;
      for (int j = 0; j < Wmax; ++j) {
        const bool on = j < Wm;
        const int m = on ? m_lo + j : m_lo;
        const double xd = fr - (double)(m - kfl);                       // x = f_n/DF - m, exact
        const float x = (float)xd;
        // the two large phases, in turns, reduced in fp64
        double th = (xd + 1.0) * (xd + 1.0) * inv2k, tl = (xd - 1.0) * (xd - 1.0) * inv2k;
        th -= floor(th);
        tl -= floor(tl);
        float sh, ch, sl, cl;
        __sincosf(6.283185307179586f * ((float)th - 0.5f), &sh, &ch);   // = -(sin, cos)(2 pi th)
        __sincosf(6.283185307179586f * ((float)tl - 0.5f), &sl, &cl);
        const Cplx Ehi = {-ch, sh}, Elo = {-cl, sl};                    // exp(-2 pi i turns)
        const float vhp = sc * (x + 1.f - kq), vhm = sc * (x + 1.f + kq);
        const float vlp = sc * (x - 1.f - kq), vlm = sc * (x - 1.f + kq);
        const Cplx Ghp = godd(vhp, lut_lane), Ghm = godd(vhm, lut_lane), Glp = godd(vlp, lut_lane), Glm = godd(vlm, lut_lane);
        const Cplx dH = {Ghp.r - Ghm.r, -(Ghp.i - Ghm.i)};              // conj(Godd(v_hi,+) - Godd(v_hi,-))
        const Cplx dL = {Glp.r - Glm.r, -(Glp.i - Glm.i)};
        Cplx rip = cmulf(Ehi, dH);
        const Cplx rl = cmulf(Elo, dL);
        rip.r += rl.r; rip.i += rl.i;
        // times exp(-i pi/4) / (2 sqrt2) = (1 - i)/4
        Cplx K = {0.25f * (rip.r + rip.i), 0.25f * (rip.i - rip.r)};
        float sx, cx;
        __sincosf(1.5707963267948966f * x, &sx, &cx);
        const float inp = (vlp < 0.f && vhp > 0.f) ? 0.5f : 0.f, inm = (vlm < 0.f && vhm > 0.f) ? 0.5f : 0.f;
        const Cplx mn = {(inp + inm) * cx, (inm - inp) * sx};           // in_+ exp(-i pi x/2) + in_- exp(+i pi x/2), halved
        const Cplx mk = cmulf(eK, mn);
        K.r += mk.r; K.i += mk.i;
        // parity factor eps_nm
        if ((n_pix + m) & 1) {
          const float sg = (n_pix & m & 1) ? -1.f : 1.f;
          K = {-sg * K.i, sg * K.r};
        }
        if (!on) K = {0.f, 0.f};
        const long long idx = (long long)m * a.ncol + col;
        const float2 y = __ldg(gy + idx), w = __ldg(gw + idx);
        z0.r = fmaf(y.x, K.r, z0.r); z0.i = fmaf(y.x, K.i, z0.i);
        z1.r = fmaf(y.y, K.r, z1.r); z1.i = fmaf(y.y, K.i, z1.i);
        const float k2 = fmaf(K.r, K.r, K.i * K.i), kr2 = fmaf(K.r, K.r, -K.i * K.i), ki2 = 2.f * K.r * K.i;
        S00 = fmaf(w.x, k2, S00); S01 = fmaf(w.y, k2, S01);
        S20.r = fmaf(w.x, kr2, S20.r); S20.i = fmaf(w.x, ki2, S20.i);
        S21.r = fmaf(w.y, kr2, S21.r); S21.i = fmaf(w.y, ki2, S21.i);
      }
      // transfer factors and the pixel's factor P = (A/sqrt2) exp(i Phi_n):  Y_alpha = T_alpha P eps K
      const Cplx TP0 = cmulf({T.T0r, T.T0i}, P), TP1 = cmulf({T.T1r, T.T1i}, P);
      const Cplx a0 = cmulf(TP0, z0), a1 = cmulf(TP1, z1);
      v[0] = a0.r + a1.r;
      v[1] = a0.i + a1.i;
      const Cplx q0 = cmulf(cmulf(TP0, TP0), S20), q1 = cmulf(cmulf(TP1, TP1), S21);
      const float n0 = (TP0.r * TP0.r + TP0.i * TP0.i) * S00 + (TP1.r * TP1.r + TP1.i * TP1.i) * S01;
      v[2] = 0.5f * (n0 + q0.r + q1.r);                                 // sum W Re(Y)^2
      v[3] = 0.5f * (n0 - q0.r - q1.r);                                 // sum W Im(Y)^2
      v[4] = 0.5f * (q0.i + q1.i);                                      // sum W Re(Y) Im(Y)
      if (!closes) {
#pragma unroll
        for (int q = 0; q < 5; ++q) acc[q] += v[q];
      }
    }
    if (closes) {
      int lo = 0;
      for (;;) {
        const bool ends = p < p_stop && pend <= cend;
        const int hi = ends ? pend - ic : 32;
        if (lane >= lo && lane < hi) {
#pragma unroll
          for (int q = 0; q < 5; ++q) acc[q] += v[q];
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

__global__ void __launch_bounds__(kWarpsPerCta * 32, 1)
eval_wdm_kernel(const EvalArgs a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float4* s_lut = reinterpret_cast<float4*>(smem_raw);
  const int lane = threadIdx.x & 31;
  for (int i = threadIdx.x; i < (kLutN + 1) * kLutCopiesList; i += blockDim.x) s_lut[i] = a.lut[i / kLutCopiesList];
  __syncthreads();
  const unsigned lut_lane = (unsigned)__cvta_generic_to_shared(s_lut) + 16u * (unsigned)(lane & (kLutCopiesList - 1)) -
                            kMagicBits * (16u * kLutCopiesList);
  const int n_units = a.n_units[1];
  for (;;) {
    unsigned long long uid = 0;
    if (lane == 0) uid = atomicAdd(a.work_counter + 1, 1ULL);
    uid = __shfl_sync(0xffffffffu, uid, 0);
    if (uid >= (unsigned long long)n_units) break;
    const Unit d = a.units_list[uid];
    for (int k = 0; k < d.cnt; ++k) eval_item_wdm(a, (long long)a.list[d.off + (unsigned)k], d.tile, lane, lut_lane);
  }
}

// P_n = [a b] G^-1 [a b]^T per segment (fp64), Upsilon = sum_n P_n; seg_dh = (a, b), seg_hh = (hcc + hss)/2
__global__ void combine_wdm_kernel(const float4* __restrict__ partials, const uint16_t* __restrict__ keys, long long n, int N_seg,
                                   const int* __restrict__ tile_first, int n_tiles, const int* __restrict__ piece_seg,
                                   const int* __restrict__ piece_tile, float* __restrict__ upsilon,
                                   float* __restrict__ seg_power, float* __restrict__ seg_dh, float* __restrict__ seg_hh) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int n_pieces = tile_first[n_tiles];
  double ups = 0.0;
  int p = 0, cur_tile = -1;
  bool live = false;
  for (int s = 0; s < N_seg; ++s) {
    double sa = 0, sb = 0, hcc = 0, hss = 0, hcs = 0;
    for (; p < n_pieces && piece_seg[p] == s; ++p) {
      const int t = piece_tile[p];
      if (t != cur_tile) { cur_tile = t; live = keys[(size_t)t * n + i] != 0; }
      if (!live) continue;
      const float4 u = partials[((long long)p * n + i) * 2], w = partials[((long long)p * n + i) * 2 + 1];
      sa += u.x; sb += u.y; hcc += u.z; hss += u.w; hcs += w.x;
    }
    const double det = hcc * hss - hcs * hcs;
    const double P = det > 0.0 ? (sa * sa * hss - 2.0 * sa * sb * hcs + sb * sb * hcc) / det : 0.0;
    ups += P;
    if (seg_power) seg_power[i * N_seg + s] = (float)P;
    if (seg_dh) { seg_dh[(i * N_seg + s) * 2] = (float)sa; seg_dh[(i * N_seg + s) * 2 + 1] = (float)sb; }
    if (seg_hh) seg_hh[i * N_seg + s] = (float)(0.5 * (hcc + hss));
  }
  upsilon[i] = (float)ups;
}

// Upload: y = W d and W interleaved by channel, transposed to [m][i] over the valid time pixels
__global__ void __launch_bounds__(256)
pack_wdm_kernel(const float* __restrict__ coeff, const float* __restrict__ weight, int Nt, int Nf, int C,
                const uint8_t* __restrict__ gap, const int* __restrict__ vprefix, int ncol,
                float2* __restrict__ gy, float2* __restrict__ gw) {
  __shared__ float2 sY[32][33];
  __shared__ float2 sW[32][33];
  const int k0 = blockIdx.x * 32, m0 = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const long long npix = (long long)Nt * Nf;
  for (int r = ty; r < 32; r += 8) {
    const int n = m0 + r, k = k0 + tx;
    if (n < Nt && k < Nf) {
      const long long i = (long long)n * Nf + k;
      float d0 = coeff[i], d1 = C > 1 ? coeff[npix + i] : 0.f;
      float w0 = weight ? weight[i] : 1.f, w1 = C > 1 ? (weight ? weight[npix + i] : 1.f) : 0.f;
      if (!(isfinite(w0 * d0) && isfinite(w0))) { w0 = 0.f; d0 = 0.f; }
      if (!(isfinite(w1 * d1) && isfinite(w1))) { w1 = 0.f; d1 = 0.f; }
      sY[r][tx] = make_float2(w0 * d0, w1 * d1);
      sW[r][tx] = make_float2(w0, w1);
    }
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const int k = k0 + r, n = m0 + tx;
    if (n < Nt && k < Nf && gap[n] != 0) {
      const long long o = (long long)k * ncol + vprefix[n];
      gy[o] = sY[tx][r];
      gw[o] = sW[tx][r];
    }
  }
}

// window pixel counts in the WDM basis
__global__ void count_pixels_wdm_kernel(const EvalArgs a, long long* __restrict__ counts) {
  const int lane = threadIdx.x & 31;
  const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= a.n) return;
  const TplConst T = load_template(a.params + w * 8, a.DT, -1, 0);
  long long cnt = 0;
  if (T.ok) {
    for (int n = lane; n < a.Nt; n += 32) {
      const TrackPoint tp = track_point_at(T, (double)n * a.wdm_DTpix, a.DT, a.x_lo, a.x_hi, a.c_max, 0.5, a.gap[n] != 0);
      if (tp.active) {
        const int kfl = __double2int_rd(tp.x);
        const int kce = tp.x > (double)kfl ? kfl + 1 : kfl;
        const int m_lo = min(max(kce - 1 - a.wdm_Hw, 1), a.Nf - 1), m_hi = min(kfl + 1 + a.wdm_Hw, a.Nf - 1);
        cnt += max(m_hi - m_lo + 1, 0);
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  if (lane == 0) counts[w] = cnt;
}

}  // namespace tfs
