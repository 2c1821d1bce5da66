// tfs_frontend.cuh -- time-series -> time-frequency front end.
// "Each tranche is Tukey-windowed with a shape parameter of 0.1 and fast-Fourier-transformed to
// construct the time-frequency grid"; tranches that overlap a gap are dropped.
//
//   D[alpha,m,k] = (1/N) sum_n w[n] x[alpha, m N + n] exp(-2 pi i k n / N),  N = 2 Nf,  k = 0 ... Nf-1
//
// One CTA per (tranche, channel).  The real series of N samples is packed as L = Nf complex numbers
// z[n] = w x[2n] + i w x[2n+1], transformed by a shared-memory Stockham FFT (radices 4, 2, 3, 5, twiddles
// from a table built in fp64) and unpacked:  X[k] = E[k] - i exp(-2 pi i k/N) O[k],
// E = (Z[k] + conj Z[L-k])/2,  O = (Z[k] - conj Z[L-k])/2.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tfs {

constexpr int kFeMaxStages = 24;
// radices of the stages, and for each stage the offset of its twiddle block in the table: stage s (radix R,
// Ns = product of the earlier radices) owns (R-1)*Ns entries, entry (t-1)*Ns + k = exp(-2 pi i t k / (Ns R)),
// so that consecutive butterflies (consecutive k) read consecutive twiddles
struct FeRadices { int n; int r[kFeMaxStages]; int off[kFeMaxStages]; int total; };

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// per-stage twiddle blocks (see FeRadices) and win[n] = Tukey(N, alpha)[n] (symmetric form), both from fp64
__global__ void fe_tables_kernel(float2* __restrict__ tw, const FeRadices rad, float* __restrict__ win, int N,
                                 double alpha) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < rad.total) {
    int st = 0, Ns = 1;
    while (st + 1 < rad.n && i >= rad.off[st + 1]) { Ns *= rad.r[st]; ++st; }
    const int e = i - rad.off[st];
    const int t = e / Ns + 1, k = e - (t - 1) * Ns;
    double s, c;
    sincospi(-2.0 * (double)t * (double)k / ((double)Ns * (double)rad.r[st]), &s, &c);
    tw[i] = make_float2((float)c, (float)s);
  }
  if (i < N) {
    double w = 1.0;
    if (N > 1 && alpha > 0.0) {
      const double edge = fmin(alpha, 1.0) * (double)(N - 1) * 0.5;
      const double n = (double)i, nr = (double)(N - 1 - i);
      if (n < edge) w = 0.5 * (1.0 - cospi(n / edge));
      else if (nr < edge) w = 0.5 * (1.0 - cospi(nr / edge));
    }
    win[i] = (float)w;
  }
}

template <int R>
__device__ __forceinline__ void small_dft(float2* v) {
  if (R == 2) {
    const float2 a = v[0], b = v[1];
    v[0] = make_float2(a.x + b.x, a.y + b.y);
    v[1] = make_float2(a.x - b.x, a.y - b.y);
  } else if (R == 4) {
    const float2 a = make_float2(v[0].x + v[2].x, v[0].y + v[2].y), b = make_float2(v[0].x - v[2].x, v[0].y - v[2].y);
    const float2 c = make_float2(v[1].x + v[3].x, v[1].y + v[3].y), d = make_float2(v[1].x - v[3].x, v[1].y - v[3].y);
    v[0] = make_float2(a.x + c.x, a.y + c.y);
    v[2] = make_float2(a.x - c.x, a.y - c.y);
    v[1] = make_float2(b.x + d.y, b.y - d.x);          // b - i d
    v[3] = make_float2(b.x - d.y, b.y + d.x);          // b + i d
  } else if (R == 3) {
    const float s = 0.86602540378443864676f;           // sin(2 pi / 3)
    const float2 t = make_float2(v[1].x + v[2].x, v[1].y + v[2].y), d = make_float2(v[1].x - v[2].x, v[1].y - v[2].y);
    const float2 m = make_float2(v[0].x - 0.5f * t.x, v[0].y - 0.5f * t.y);
    v[0] = make_float2(v[0].x + t.x, v[0].y + t.y);
    v[1] = make_float2(m.x + s * d.y, m.y - s * d.x);  // m - i s d
    v[2] = make_float2(m.x - s * d.y, m.y + s * d.x);  // m + i s d
  } else {   // R == 5
    const float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f;   // cos(2 pi/5), cos(4 pi/5)
    const float s1 = 0.95105651629515357212f, s2 = 0.58778525229247312917f;    // sin(2 pi/5), sin(4 pi/5)
    const float2 a1 = make_float2(v[1].x + v[4].x, v[1].y + v[4].y), b1 = make_float2(v[1].x - v[4].x, v[1].y - v[4].y);
    const float2 a2 = make_float2(v[2].x + v[3].x, v[2].y + v[3].y), b2 = make_float2(v[2].x - v[3].x, v[2].y - v[3].y);
    const float2 v0 = v[0];
    v[0] = make_float2(v0.x + a1.x + a2.x, v0.y + a1.y + a2.y);
    const float2 p1 = make_float2(v0.x + c1 * a1.x + c2 * a2.x, v0.y + c1 * a1.y + c2 * a2.y);
    const float2 p2 = make_float2(v0.x + c2 * a1.x + c1 * a2.x, v0.y + c2 * a1.y + c1 * a2.y);
    const float2 q1 = make_float2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y);
    const float2 q2 = make_float2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y);
    v[1] = make_float2(p1.x + q1.y, p1.y - q1.x);      // p1 - i q1
    v[4] = make_float2(p1.x - q1.y, p1.y + q1.x);
    v[2] = make_float2(p2.x + q2.y, p2.y - q2.x);
    v[3] = make_float2(p2.x - q2.y, p2.y + q2.x);
  }
}

// shared-memory index swizzle: XOR the low 4 bits with the next 4.  Consecutive elements stay a permutation
// of their aligned block of 16 (conflict-free loads), while the strided stores of the first stages
// (out[4 j + t], out[16 a + b + 4 t]) spread over the banks: 2304 -> 1344 store wavefronts per transform at
// L = 3072 (1152 is the minimum).  smask = 15 when L is a multiple of 16, else 0 (no swizzle).
__device__ __forceinline__ int fe_swz(int e, int smask) { return e ^ ((e >> 4) & smask); }

// one Stockham stage of radix R: Ns = product of the radices of the stages already done, tw = this stage's
// twiddle block
template <int R>
__device__ __forceinline__ void stockham_stage(const float2* __restrict__ in, float2* __restrict__ out, int L, int Ns,
                                               const float2* __restrict__ tw, int smask) {
  const int LR = L / R;
  const bool pow2 = (Ns & (Ns - 1)) == 0;        // the host puts the odd radices last, so this is the usual case
  for (int j = threadIdx.x; j < LR; j += blockDim.x) {
    const int k = pow2 ? (j & (Ns - 1)) : (j % Ns);
    float2 v[R];
#pragma unroll
    for (int t = 0; t < R; ++t) {
      v[t] = in[fe_swz(j + t * LR, smask)];
      if (t > 0) v[t] = cmul(v[t], __ldg(tw + (t - 1) * Ns + k));
    }
    small_dft<R>(v);
    const int j0 = (j - k) * R + k;
#pragma unroll
    for (int t = 0; t < R; ++t) out[fe_swz(j0 + t * Ns, smask)] = v[t];
  }
}

// grid (Nt, C), dynamic shared memory 2 * L * sizeof(float2) (the twiddle table stays in global memory / L2:
// a copy in shared memory costs occupancy and measured 13 % slower)
#ifndef TFS_FE_THREADS
#define TFS_FE_THREADS 512
#endif
constexpr int kFeThreads = TFS_FE_THREADS;
__global__ void __launch_bounds__(kFeThreads)
fe_fft_kernel(const float* __restrict__ x, const float* __restrict__ win, const float2* __restrict__ tw,
              const FeRadices rad, int Nt, int Nf, float2* __restrict__ coeff_out, uint8_t* __restrict__ gap) {
  extern __shared__ float2 fe_smem[];
  const int L = Nf, N = 2 * Nf;
  const int m = blockIdx.x, a = blockIdx.y;
  float2* cur = fe_smem;
  float2* nxt = fe_smem + L;
  const float2* xs = reinterpret_cast<const float2*>(x + ((size_t)a * Nt + m) * N);      // N is even: 8-byte aligned
  const float2* ws = reinterpret_cast<const float2*>(win);
  const int smask = (L & 15) == 0 ? 15 : 0;
  int bad = 0;
  for (int n = threadIdx.x; n < L; n += blockDim.x) {
    const float2 s = __ldg(xs + n), w = __ldg(ws + n);
    bad |= !(isfinite(s.x) && isfinite(s.y));
    cur[fe_swz(n, smask)] = make_float2(s.x * w.x, s.y * w.y);
  }
  // a tranche with a sample that is not finite carries no usable transform: it is dropped like a gap (C20)
  if (__syncthreads_or(bad) && threadIdx.x == 0 && gap) gap[m] = 0;
  int Ns = 1;
  for (int st = 0; st < rad.n; ++st) {
    const int R = rad.r[st];
    if (R == 4) stockham_stage<4>(cur, nxt, L, Ns, tw + rad.off[st], smask);
    else if (R == 2) stockham_stage<2>(cur, nxt, L, Ns, tw + rad.off[st], smask);
    else if (R == 3) stockham_stage<3>(cur, nxt, L, Ns, tw + rad.off[st], smask);
    else stockham_stage<5>(cur, nxt, L, Ns, tw + rad.off[st], smask);
    Ns *= R;
    __syncthreads();
    float2* t = cur; cur = nxt; nxt = t;
  }
  const float invN = 1.0f / (float)N;
  float2* out = coeff_out + ((size_t)a * Nt + m) * Nf;
  for (int k = threadIdx.x; k < L; k += blockDim.x) {
    const float2 zk = cur[fe_swz(k, smask)], zc = cur[fe_swz(k == 0 ? 0 : L - k, smask)];
    const float2 E = make_float2(0.5f * (zk.x + zc.x), 0.5f * (zk.y - zc.y));      // (Z[k] + conj Z[L-k]) / 2
    const float2 O = make_float2(0.5f * (zk.x - zc.x), 0.5f * (zk.y + zc.y));      // (Z[k] - conj Z[L-k]) / 2
    float s, c;
    sincospif(-(float)k / (float)L, &s, &c);                                        // exp(-2 pi i k / N)
    const float2 tO = cmul(make_float2(c, s), O);
    out[k] = make_float2((E.x + tO.y) * invN, (E.y - tO.x) * invN);                // E - i tO
  }
}

// W[alpha,m,k] = 4 DT / S_alpha[k] (0 where S is not positive and finite), or 1 without a PSD; grid (k blocks, Nt, C)
__global__ void fe_weight_kernel(const float* __restrict__ psd, int Nt, int Nf, double DT, float* __restrict__ weight_out) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y, a = blockIdx.z;
  if (k >= Nf) return;
  float w = 1.0f;
  if (psd) {
    const float S = psd[(size_t)a * Nf + k];
    w = (isfinite(S) && S > 0.0f) ? (float)(4.0 * DT / (double)S) : 0.0f;
  }
  weight_out[((size_t)a * Nt + m) * Nf + k] = w;
}

// b[alpha][k] = 4 DT / S_alpha[k] (0 where S is not positive and finite): the per-bin weight table of the front end
__global__ void fe_bk_kernel(const float* __restrict__ psd, int C, int Nf, double DT, float* __restrict__ bk) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= C * Nf) return;
  const float S = psd[i];
  bk[i] = (isfinite(S) && S > 0.0f) ? (float)(4.0 * DT / (double)S) : 0.0f;
}

// g[m] = 1 iff every sample of tranche m is valid; one block per tranche
__global__ void __launch_bounds__(256)
fe_gap_kernel(const uint8_t* __restrict__ sample_mask, int N, uint8_t* __restrict__ gap_out) {
  const int m = blockIdx.x;
  int bad = 0;
  if (sample_mask) {
    const uint8_t* row = sample_mask + (size_t)m * N;
    if ((N & 15) == 0 && (((uintptr_t)row) & 15) == 0) {
      // 16 mask bytes per load: a zero byte anywhere in the word (the classic has-zero-byte test)
      const uint4* r4 = reinterpret_cast<const uint4*>(row);
      for (int n = threadIdx.x; n < N / 16; n += blockDim.x) {
        const uint4 v = __ldg(r4 + n);
        const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int q = 0; q < 4; ++q) bad |= ((w[q] - 0x01010101u) & ~w[q] & 0x80808080u) != 0u;
      }
    } else {
      for (int n = threadIdx.x; n < N; n += blockDim.x) bad |= (row[n] == 0);
    }
  }
  bad = __syncthreads_or(bad);
  if (threadIdx.x == 0) gap_out[m] = bad ? 0 : 1;
}

}  // namespace tfs
