// tfs.cu -- host side of libtfs: C ABI (include/tfs.h), context, launches.
// No torch, no third-party libraries: CUDA runtime only.
#include "../../include/tfs.h"
#include "tfs_kernels.cuh"
#include "tfs_frontend.cuh"
#include "tfs_wdm.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

using namespace tfs;

namespace {

thread_local char g_create_err[512] = "";

constexpr size_t kScratchBytes = 2ull << 30;  // cap for the piece-partials buffer per sub-batch

}  // namespace

// FP32 issue probe (tfs_probe_fp32_issue): one 1024-thread CTA per SM, every thread runs kProbeChains independent
// chains of dependent fused multiply-adds -- scalar FFMA, or packed FFMA2 (fma.rn.f32x2, the instruction the pixel loops
// are made of) -- and the CTA's duration is read from the SM's own cycle counter.
constexpr int kProbeChains = 8;
__global__ void __launch_bounds__(1024, 1) fp32_issue_probe_kernel(int iters, int packed, float* sink, unsigned long long* cycles) {
  const float x = 1.0f + 1e-7f * (float)threadIdx.x, y = 1e-9f * (float)(blockIdx.x + 1);
  float acc = 0.f;
  __syncthreads();
  const long long t0 = clock64();
  if (packed) {
    f2_t v[kProbeChains];
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) v[c] = pk((float)c, (float)c + 0.5f);
    const f2_t m = pk(x, x), b = pk(y, y);
#pragma unroll 4
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int c = 0; c < kProbeChains; ++c) v[c] = ffma2(v[c], m, b);
    }
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) { float lo, hi; upk(v[c], lo, hi); acc += lo + hi; }
  } else {
    float v[kProbeChains];
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) v[c] = (float)c;
#pragma unroll 4
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int c = 0; c < kProbeChains; ++c) v[c] = fmaf(v[c], x, y);
    }
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) acc += v[c];
  }
  __syncthreads();
  const long long t1 = clock64();
  if (threadIdx.x == 0) cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
  if (acc == 123.456f) *sink = acc;      // keeps the chains alive
}

struct tfs_ctx {
  int Nt = 0, Nf = 0, C = 0;
  double dt = 0, DT = 0, df = 0;
  tfs_opts opts{};
  double f_lo = 0, f_hi = 0;
  int device = 0, sm_count = 0;
  bool uploaded = false;

  // channel pairs: pair 0 = channels (0, 1), pair 1 = channel 2 (n_channels = 3); a missing half is zeros
  struct Pair {
    float4* grid = nullptr;                // [Nf + kPadRows][ncol_cap]
    float2* wgt = nullptr;
    float2* wa = nullptr;                  // [ncol_cap] separable weights: a[i] by valid-tranche index
    float2* wb = nullptr;                  // [Nf + kPadRows + kSlabRowsMax] separable weights: b[k]
    int c0 = 0, c1 = -1;                   // channels packed in the pair (-1: empty half)
    CUtensorMap map_y, map_w;              // TMA descriptors of grid / wgt for the slab kernel (set at upload)
  } pair[2];
  int n_pairs = 1;
  int ncol_cap = 0, ncol = 0;              // columns allocated per row (Nt rounded up to kTS), columns in use
  float2* colmax = nullptr;                // [Nf] scratch of the weight analysis
  unsigned long long* wcounts = nullptr;   // [2] {pixels violating W = a b, columns with b != 1}
  bool t3_set = false;                     // tfs_set_third_channel_factor was called (3-channel contexts)
  double t3[2] = {0.0, 0.0};               // constant T_T of the third channel for tfs_eval / tfs_eval_tseg
  int wmode = -1;                          // kWGeneral / kWSeparable / kWTimeOnly; -1 before the first upload
  int n_valid = 0;                         // valid (non-gap) tranches of the data uploaded last
  // piece tables (tile x segment cuts of the valid-tranche list), cached per N_seg until the next upload
  struct PieceTable { int N_seg; int M_tr; int n_tiles; int* tile_first; int* piece_end; int* piece_seg; int* piece_tile; cudaEvent_t ready; };
  std::vector<PieceTable> piece_tables;
  uint8_t* gap = nullptr;
  int* vprefix = nullptr;                  // [Nt+1] valid tranches before m
  int* valid_m = nullptr;                  // [max(#valid,1)] valid tranche indices
  float4* lut = nullptr;
  FarCoef far{};
  unsigned long long* bad = nullptr;       // device counter
  unsigned long long* work = nullptr;      // [2] device unit counters of the slab and the list kernel
  unsigned long long* census = nullptr;    // [5] device tier counters (tfs_tier_census); handed to the kernels only while census_on
  bool census_on = false;
  long long bad_host = 0;

  // growable device scratch
  void* buf_params = nullptr;   size_t cap_params = 0;
  void* buf_partials = nullptr; size_t cap_partials = 0;
  void* buf_prep = nullptr;     size_t cap_prep = 0;      // per-batch pre-pass: constants, keys, bucket tables, lists, units
  void* buf_ttab = nullptr;     size_t cap_ttab = 0;      // staged transfer table (tfs_eval_tf with a host table)
  void* buf_out[5] = {nullptr, nullptr, nullptr, nullptr, nullptr}; size_t cap_out[5] = {0, 0, 0, 0, 0};
  void* buf_keys = nullptr;     size_t cap_keys = 0;
  void* buf_tk_in = nullptr;    size_t cap_tk_in = 0;
  void* buf_tk_idx = nullptr;   size_t cap_tk_idx = 0;
  void* buf_tk_val = nullptr;   size_t cap_tk_val = 0;
  void* buf_counts = nullptr;   size_t cap_counts = 0;
  void* buf_children = nullptr; size_t cap_children = 0;
  void* buf_fe = nullptr;       size_t cap_fe = 0;        // front-end temporaries (tfs_upload_timeseries)
  SelectState* sel = nullptr;

  // measurement hooks
  bool profiling = false;
  std::vector<cudaEvent_t> ev_pool;        // reused events, three per evaluation launch: start, list kernel done, slab kernel done
  size_t ev_used = 0;
  long long launches = 0;
  long long l2_window_used = 0;            // evaluation launches that ran under an L2 access-policy window (TFS_L2_WINDOW=1)

  char err[512] = "";
};

namespace {

int fail(tfs_ctx* ctx, int code, const char* fmt, ...) {
  char* dst = ctx ? ctx->err : g_create_err;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 512, fmt, ap);
  va_end(ap);
  return code;
}

#define TFS_CUDA(ctx, expr)                                                              \
  do {                                                                                   \
    cudaError_t e_ = (expr);                                                             \
    if (e_ != cudaSuccess) {                                                             \
      const int code_ = (e_ == cudaErrorMemoryAllocation) ? TFS_ENOMEM : TFS_ECUDA;      \
      return fail(ctx, code_, "%s failed: %s", #expr, cudaGetErrorString(e_));           \
    }                                                                                    \
  } while (0)

// true if p is device-accessible memory (device or managed); host (pageable/pinned) otherwise
bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  cudaError_t e = cudaPointerGetAttributes(&at, p);
  if (e != cudaSuccess) { cudaGetLastError(); return false; }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

int ensure(tfs_ctx* ctx, void** buf, size_t* cap, size_t bytes) {
  if (*cap >= bytes) return TFS_OK;
  if (*buf) { cudaFree(*buf); *buf = nullptr; *cap = 0; }
  const size_t want = bytes + bytes / 8;
  cudaError_t e = cudaMalloc(buf, want);
  if (e != cudaSuccess) {
    cudaGetLastError();
    e = cudaMalloc(buf, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, TFS_ENOMEM, "cudaMalloc(%zu bytes) failed", bytes); }
    *cap = bytes;
    return TFS_OK;
  }
  *cap = want;
  return TFS_OK;
}

// ---------------------------------------------------------------------------------------------
// Host-side Fresnel auxiliary functions f(v), g(v) (A&S 7.3.5-6; ref [52] of the paper) for the LUT.
//   v <= 5.5 : C(v), S(v) by composite Gauss-Legendre quadrature of the defining integrals
//   v  > 5.5 : asymptotic series (DLMF 7.12.2-3; ref [53] of the paper)
// ---------------------------------------------------------------------------------------------
struct GaussLegendre {
  static constexpr int N = 16;
  double x[N], w[N];
  GaussLegendre() {
    for (int i = 0; i < N; ++i) {
      double z = std::cos(kPi * (i + 0.75) / (N + 0.5));
      double pp = 1.0;
      for (int it = 0; it < 100; ++it) {
        double p1 = 1.0, p2 = 0.0;
        for (int j = 1; j <= N; ++j) { double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
        pp = N * (z * p1 - p2) / (z * z - 1.0);
        const double dz = p1 / pp;
        z -= dz;
        if (std::fabs(dz) < 1e-16) break;
      }
      x[i] = z;
      w[i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
  }
};

void fresnel_cs_quadrature(double v, double& C, double& S) {
  static const GaussLegendre gl;
  C = 0.0; S = 0.0;
  const int panels = std::max(1, (int)std::ceil(v / 0.125));
  const double h = v / panels;
  for (int p = 0; p < panels; ++p) {
    const double a = p * h, mid = a + 0.5 * h;
    for (int i = 0; i < GaussLegendre::N; ++i) {
      const double t = mid + 0.5 * h * gl.x[i];
      const double ph = 0.5 * kPi * t * t;
      C += 0.5 * h * gl.w[i] * std::cos(ph);
      S += 0.5 * h * gl.w[i] * std::sin(ph);
    }
  }
}

void fresnel_aux_host(double v, double& f, double& g) {
  if (v <= 5.5) {
    double C, S;
    fresnel_cs_quadrature(v, C, S);
    const double a = 0.5 * kPi * std::fmod(v * v, 4.0);
    f = (0.5 - S) * std::cos(a) - (0.5 - C) * std::sin(a);
    g = (0.5 - C) * std::cos(a) + (0.5 - S) * std::sin(a);
    return;
  }
  const double w = 0.5 * kPi * v * v;
  double sf = 0.0, sg = 0.0, poch = 1.0, wp = 1.0, last = 1e300, sign = 1.0;   // poch = (1/2)_{2m}, wp = w^{2m}
  for (int m = 0; m < 200; ++m) {
    const double tf = poch / wp;
    if (tf > last || tf < 1e-20) break;
    last = tf;
    const double tg = poch * (0.5 + 2 * m) / (wp * w);
    sf += sign * tf;
    sg += sign * tg;
    poch *= (0.5 + 2 * m) * (1.5 + 2 * m);
    wp *= w * w;
    sign = -sign;
  }
  f = sf / (kPi * v);
  g = sg / (kPi * v);
}

void build_lut(std::vector<float4>& lut) {
  // F = f/t, G = g/t at t_i = i/kLutN (v_i = 1/t_i - 1), two extra nodes past each end for the slopes
  auto node = [](int i, double& F, double& G) {
    if (i <= 0) { F = 1.0 / kPi; G = 0.0; return; }         // t -> 0: f/t = f (1+v) -> 1/pi ; g/t -> 0
    const double t = (double)i / kLutN;
    const double v = std::max(1.0 / t - 1.0, 0.0);
    double f, g;
    fresnel_aux_host(v, f, g);
    F = f / t;
    G = g / t;
  };
  lut.resize(kLutN + 1);
  for (int i = 0; i <= kLutN; ++i) {
    double F, G, Fm, Gm, Fp, Gp;
    node(i, F, G);
    const int im = std::max(i - 1, 0), ip = std::min(i + 1, kLutN);
    node(im, Fm, Gm);
    node(ip, Fp, Gp);
    const double w = (double)(ip - im);                      // central difference (one-sided at the ends)
    // interpolant around node i as intercept + slope * t:  F(t) ~ F_i + (t kLutN - i) dF  (see fresnel_aux)
    const double dF = (Fp - Fm) / w, dG = (Gp - Gm) / w;
    lut[i] = make_float4((float)(G - i * dG), (float)(F - i * dF), (float)(kLutN * dG), (float)(kLutN * dF));
  }
}

// Far-zone polynomials (kernel: pixel_far).  For v >= kVFar,
//   f(v) = w (1/pi + F1 z + F2 z^2),  g(v) = w^3 (1/pi^2 + G1 z + G2 z^2),  w = 1/v, z = w^4
// -- the shape of the asymptotic series A&S 7.3.27-28 (f ~ 1/(pi v) - 3/(pi^3 v^5) + ...,
// g ~ 1/(pi^2 v^3) - 15/(pi^4 v^7) + ...): the leading coefficients are kept exact, so the relative error
// vanishes as v grows (slow chirps put their brightest pixels at v ~ 5...40), and the other two are
// fitted by least squares on Chebyshev nodes of z in [0, z_max], weighted so that the error RELATIVE to
// |g + i f| ~ f is minimised.  Returns the largest such relative error over the nodes.
double fit_far(FarCoef& out) {
  const int N = 256;
  const double v_min = (double)kVFar * 0.98;
  const double z_max = 1.0 / (v_min * v_min * v_min * v_min);
  const double F0 = 1.0 / kPi, G0 = 1.0 / (kPi * kPi);
  double Af[2][3] = {{0}}, Ag[2][3] = {{0}};        // normal equations in the scaled variable y = z/z_max
  std::vector<double> ys(N), w1(N), tf(N), tg(N);
  for (int i = 0; i < N; ++i) {
    const double y = std::max(0.5 * (1.0 + std::cos(kPi * (i + 0.5) / N)), 1e-9);
    const double z = y * z_max, w = std::sqrt(std::sqrt(z)), v = 1.0 / w;
    double f, g;
    fresnel_aux_host(v, f, g);
    ys[i] = y; w1[i] = w; tf[i] = f; tg[i] = g;
    // residuals divided by f:  (w (F0 + y a1 + y^2 a2) - f)/f  and  (w^3 (G0 + y b1 + y^2 b2) - g)/f
    const double sf = w / f, sg = w * w * w / f;
    const double b[2] = {y, y * y};
    const double rf = (f - w * F0) / f, rg = (g - w * w * w * G0) / f;
    for (int r = 0; r < 2; ++r) {
      for (int c = 0; c < 2; ++c) { Af[r][c] += sf * b[r] * sf * b[c]; Ag[r][c] += sg * b[r] * sg * b[c]; }
      Af[r][2] += sf * b[r] * rf;
      Ag[r][2] += sg * b[r] * rg;
    }
  }
  auto solve2 = [](double A[2][3], double x[2]) {
    const double det = A[0][0] * A[1][1] - A[0][1] * A[1][0];
    x[0] = (A[0][2] * A[1][1] - A[0][1] * A[1][2]) / det;
    x[1] = (A[0][0] * A[1][2] - A[0][2] * A[1][0]) / det;
  };
  double cf[2], cg[2];
  solve2(Af, cf);
  solve2(Ag, cg);
  double err = 0.0;
  for (int i = 0; i < N; ++i) {
    const double y = ys[i], w = w1[i];
    err = std::max(err, std::fabs(w * (F0 + y * (cf[0] + y * cf[1])) - tf[i]) / tf[i]);
    err = std::max(err, std::fabs(w * w * w * (G0 + y * (cg[0] + y * cg[1])) - tg[i]) / tf[i]);
  }
  out.F0 = (float)F0; out.F1 = (float)(cf[0] / z_max); out.F2 = (float)(cf[1] / (z_max * z_max));
  out.G0 = (float)G0; out.G1 = (float)(cg[0] / z_max); out.G2 = (float)(cg[1] / (z_max * z_max));
  return err;
}

void free_piece_tables(tfs_ctx* ctx) {
  for (auto& t : ctx->piece_tables) {
    cudaFree(t.tile_first); cudaFree(t.piece_end); cudaFree(t.piece_seg); cudaFree(t.piece_tile);
    if (t.ready) cudaEventDestroy(t.ready);
  }
  ctx->piece_tables.clear();
}

// piece table for N_seg (built on `st` on first use; later users on other streams wait for the build event)
int get_piece_table(tfs_ctx* ctx, int N_seg, int M_tr, cudaStream_t st, const tfs_ctx::PieceTable** out) {
  for (auto& t : ctx->piece_tables)
    if (t.N_seg == N_seg && t.M_tr == M_tr) {
      // the build was synchronised when the table was made: nothing to wait for (and a tfs_eval that is being captured
      // into a CUDA graph stays free of dependencies on work outside the capture)
      *out = &t;
      return TFS_OK;
    }
  if (ctx->piece_tables.size() >= 64) free_piece_tables(ctx);         // a sweep over many N_seg: start over
  tfs_ctx::PieceTable t{};
  t.N_seg = N_seg;
  t.M_tr = M_tr;
  t.n_tiles = std::max(1, (ctx->n_valid + kTS - 1) / kTS);
  const size_t max_pieces = (size_t)t.n_tiles + (size_t)N_seg;
  cudaError_t e;
  if ((e = cudaMalloc((void**)&t.tile_first, (t.n_tiles + 1) * sizeof(int))) != cudaSuccess ||
      (e = cudaMalloc((void**)&t.piece_end, max_pieces * sizeof(int))) != cudaSuccess ||
      (e = cudaMalloc((void**)&t.piece_seg, max_pieces * sizeof(int))) != cudaSuccess ||
      (e = cudaMalloc((void**)&t.piece_tile, max_pieces * sizeof(int))) != cudaSuccess ||
      (e = cudaEventCreateWithFlags(&t.ready, cudaEventDisableTiming)) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(t.tile_first); cudaFree(t.piece_end); cudaFree(t.piece_seg); cudaFree(t.piece_tile);
    return fail(ctx, TFS_ENOMEM, "piece table allocation failed: %s", cudaGetErrorString(e));
  }
  piece_table_kernel<<<1, 1, 0, st>>>(ctx->vprefix, ctx->valid_m, ctx->Nt, N_seg, M_tr, ctx->n_valid, t.n_tiles,
                                      t.tile_first, t.piece_end, t.piece_seg, t.piece_tile);
  ctx->launches += 1;
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaEventRecord(t.ready, st);
  ctx->piece_tables.push_back(t);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);      // once per (N_seg, upload): later calls on any stream just use it
  if (e != cudaSuccess) return fail(ctx, TFS_ECUDA, "piece_table_kernel failed: %s", cudaGetErrorString(e));
  *out = &ctx->piece_tables.back();
  return TFS_OK;
}

EvalArgs base_args(const tfs_ctx* ctx, int pr = 0) {
  EvalArgs a{};
  const tfs_ctx::Pair& P = ctx->pair[pr];
  a.grid = P.grid; a.wgt = P.wgt; a.wa = P.wa; a.wb = P.wb; a.gap = ctx->gap; a.lut = ctx->lut;
  a.vprefix = ctx->vprefix; a.valid_m = ctx->valid_m;
  a.bad_count = ctx->bad;
  a.work_counter = ctx->work;
  a.census = ctx->census_on ? ctx->census : nullptr;
  a.Nt = ctx->Nt; a.Nf = ctx->Nf; a.ncol = ctx->ncol;
  a.H = ctx->opts.half_width; a.adaptive = ctx->opts.adaptive_width;
  a.DT = ctx->DT;
  a.x_lo = ctx->f_lo * ctx->DT; a.x_hi = ctx->f_hi * ctx->DT;
  a.c_max = ctx->opts.basis == 1 ? ctx->opts.wdm_kappa_max : ctx->opts.c_max;
  a.basis = ctx->opts.basis; a.wdm_Hw = ctx->opts.wdm_half_width; a.wdm_DTpix = 0.5 * ctx->DT;
  a.far = ctx->far;
  if (ctx->opts.tukey_alpha > 0.0) { a.far.win_ell = (float)(0.5 * ctx->opts.tukey_alpha); a.far.win_b = (float)(1.0 / ctx->opts.tukey_alpha); }
  a.n_valid = ctx->n_valid; a.n_tiles = 1; a.n_keys = 2;
  a.wmode = ctx->wmode;
  a.t_col = 3; a.n_ch_pair = P.c1 >= 0 ? 2 : 1;
  return a;
}

// the context's device must be current (a caller that switched devices would launch on the wrong GPU)
int check_device(tfs_ctx* ctx, const char* who) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return fail(ctx, TFS_ECUDA, "%s: cudaGetDevice failed", who); }
  if (dev != ctx->device)
    return fail(ctx, TFS_ESTATE, "%s: the context was created on device %d but device %d is current", who, ctx->device, dev);
  return TFS_OK;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 2-D TMA descriptor over a [rows][ncol] array of `floats_per_pixel` floats per pixel; box = kTS columns x box_rows rows
int encode_map(tfs_ctx* ctx, CUtensorMap* map, void* base, int floats_per_pixel, int ncol, int rows, int box_rows) {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || !p) {
      cudaGetLastError();
      return fail(ctx, TFS_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
    }
    fn = (EncodeTiledFn)p;
  }
  const cuuint64_t dims[2] = {(cuuint64_t)ncol * floats_per_pixel, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)ncol * floats_per_pixel * sizeof(float)};
  const cuuint32_t box[2] = {(cuuint32_t)(kTS * floats_per_pixel), (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(ctx, TFS_ECUDA, "cuTensorMapEncodeTiled failed with code %d", (int)r);
  return TFS_OK;
}

// params on host -> staged copy in ctx scratch; on device -> used in place
int stage_params(tfs_ctx* ctx, const double* params, long long n, cudaStream_t st, const double** d_params) {
  if (is_device_ptr(params)) { *d_params = params; return TFS_OK; }
  const size_t bytes = (size_t)n * TFS_PARAM_COLS * sizeof(double);
  int rc = ensure(ctx, &ctx->buf_params, &ctx->cap_params, bytes);
  if (rc) return rc;
  TFS_CUDA(ctx, cudaMemcpyAsync(ctx->buf_params, params, bytes, cudaMemcpyHostToDevice, st));
  *d_params = (const double*)ctx->buf_params;
  return TFS_OK;
}

}  // namespace

// =============================================================================================
extern "C" {

void tfs_default_opts(tfs_opts* o) {
  if (!o) return;
  o->half_width = 10;
  o->adaptive_width = 1;
  o->c_max = 300.0;
  o->f_lo = 0.0;
  o->f_hi = 0.0;
  o->fresnel_mode = 0;
  o->weight_mode = 0;
  o->basis = 0;
  o->wdm_half_width = 2;
  o->wdm_kappa_max = 8.0;
  o->tukey_alpha = 0.0;
}

const char* tfs_last_error(const tfs_ctx* ctx) { return ctx ? ctx->err : g_create_err; }

int tfs_weight_structure(const tfs_ctx* ctx) { return ctx ? ctx->wmode : -1; }

long long tfs_bad_param_count(const tfs_ctx* ctx) {
  if (!ctx) return 0;
  if (ctx->bad_host < 0) {
    // the last tfs_eval wrote only device outputs and did not synchronise: read the counter now
    unsigned long long bad = 0;
    if (cudaDeviceSynchronize() != cudaSuccess ||
        cudaMemcpy(&bad, ctx->bad, sizeof(bad), cudaMemcpyDeviceToHost) != cudaSuccess) {
      cudaGetLastError();
      return -1;
    }
    const_cast<tfs_ctx*>(ctx)->bad_host = (long long)bad;
  }
  return ctx->bad_host;
}

int tfs_create(tfs_ctx** out, int Nt, int Nf, double dt, int n_channels, const tfs_opts* opts) {
  if (!out) return fail(nullptr, TFS_EINVAL, "tfs_create: out is NULL");
  *out = nullptr;
  if (Nt < 1 || Nf < 2 || !(dt > 0.0) || !std::isfinite(dt))
    return fail(nullptr, TFS_EINVAL, "tfs_create: need Nt >= 1, Nf >= 2, dt > 0 (got %d, %d, %g)", Nt, Nf, dt);
  if (Nt > 2000000)        // launch grids carry Nt/32 (pack) and Nt/kTS (pre-pass) on gridDim.y (<= 65535)
    return fail(nullptr, TFS_EINVAL, "tfs_create: Nt must be <= 2000000 (got %d)", Nt);
  const int ncol_cap = (Nt + kTS - 1) / kTS * kTS;
  if ((long long)ncol_cap * (Nf + kPadRows) >= (1ll << 31))
    return fail(nullptr, TFS_EINVAL, "tfs_create: Nt*(Nf+%d) must be < 2^31", kPadRows);
  if (n_channels < 1 || n_channels > 3)
    return fail(nullptr, TFS_EINVAL, "tfs_create: n_channels must be 1, 2 or 3 (P:76-79 Eq. 3: A, E, T); got %d", n_channels);
  tfs_opts o;
  tfs_default_opts(&o);
  if (opts) o = *opts;
  if (o.half_width < 0 || o.half_width > 4096 || !(o.c_max >= 0.0) || o.c_max > 1e6 ||
      (o.fresnel_mode != 0 && o.fresnel_mode != 1) || (o.weight_mode != 0 && o.weight_mode != 1) ||
      (o.basis != 0 && o.basis != 1) || o.wdm_half_width < 0 || o.wdm_half_width > 64 || !(o.wdm_kappa_max > 0.0) ||
      o.wdm_kappa_max > 1e4)
    return fail(nullptr, TFS_EINVAL, "tfs_create: bad options (half_width %d, c_max %g, fresnel_mode %d, weight_mode %d, basis %d, "
                "wdm_half_width %d, wdm_kappa_max %g)", o.half_width, o.c_max, o.fresnel_mode, o.weight_mode, o.basis,
                o.wdm_half_width, o.wdm_kappa_max);
  if (o.basis == 1 && (n_channels > 2 || o.fresnel_mode != 0))
    return fail(nullptr, TFS_EINVAL, "tfs_create: the WDM basis takes 1 or 2 channels and fresnel_mode 0");
  if (!(o.tukey_alpha >= 0.0) || o.tukey_alpha > 1.0 || (o.tukey_alpha > 0.0 && o.tukey_alpha < 1e-3) ||
      (o.tukey_alpha > 0.0 && (o.basis != 0 || o.fresnel_mode != 0)))
    return fail(nullptr, TFS_EINVAL, "tfs_create: tukey_alpha must be 0 or in [1e-3, 1], with basis 0 and fresnel_mode 0 (got %g)",
                o.tukey_alpha);
  tfs_ctx* ctx = new (std::nothrow) tfs_ctx();
  if (!ctx) return fail(nullptr, TFS_ENOMEM, "tfs_create: host allocation failed");
  ctx->Nt = Nt; ctx->Nf = Nf; ctx->C = n_channels; ctx->dt = dt;
  ctx->DT = 2.0 * Nf * dt;
  ctx->df = 1.0 / ctx->DT;
  ctx->opts = o;
  ctx->f_lo = o.f_lo > 0.0 ? o.f_lo : ctx->df;
  ctx->f_hi = o.f_hi > 0.0 ? o.f_hi : (Nf - 1) * ctx->df;
  ctx->ncol_cap = ncol_cap;
  ctx->ncol = kTS;
  ctx->n_pairs = n_channels == 3 ? 2 : 1;
  ctx->pair[0].c0 = 0; ctx->pair[0].c1 = n_channels >= 2 ? 1 : -1;
  ctx->pair[1].c0 = 2; ctx->pair[1].c1 = -1;

  auto bail = [&](int code, const char* what, cudaError_t e) {
    fail(nullptr, code, "tfs_create: %s: %s", what, cudaGetErrorString(e));
    tfs_destroy(ctx);
    return code;
  };
  cudaError_t e = cudaGetDevice(&ctx->device);
  if (e != cudaSuccess) return bail(TFS_ECUDA, "cudaGetDevice (no CUDA device: libtfs has no CPU fallback)", e);
  e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device);
  if (e != cudaSuccess) return bail(TFS_ECUDA, "cudaDeviceGetAttribute", e);
  // kPadRows zeroed rows behind row Nf-1: the global gather may read a few pixels past a window (pixel_loop_global)
  const size_t npix = (size_t)ncol_cap * (Nf + kPadRows);
  const size_t nwb = (size_t)Nf + kPadRows + kSlabRowsMax;
  for (int pr = 0; pr < ctx->n_pairs; ++pr) {
    tfs_ctx::Pair& P = ctx->pair[pr];
    if ((e = cudaMalloc((void**)&P.grid, npix * sizeof(float4))) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc grid", e);
    if ((e = cudaMalloc((void**)&P.wgt, npix * sizeof(float2))) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc weights", e);
    if ((e = cudaMalloc((void**)&P.wa, (size_t)ncol_cap * sizeof(float2))) != cudaSuccess ||
        (e = cudaMalloc((void**)&P.wb, nwb * sizeof(float2))) != cudaSuccess)
      return bail(TFS_ENOMEM, "cudaMalloc weight factors", e);
    if ((e = cudaMemset(P.wb, 0, nwb * sizeof(float2))) != cudaSuccess) return bail(TFS_ECUDA, "cudaMemset wb", e);
  }
  if ((e = cudaMalloc((void**)&ctx->colmax, (size_t)Nf * sizeof(float2))) != cudaSuccess ||
      (e = cudaMalloc((void**)&ctx->wcounts, 2 * sizeof(unsigned long long))) != cudaSuccess)
    return bail(TFS_ENOMEM, "cudaMalloc weight analysis", e);
  if ((e = cudaMalloc((void**)&ctx->gap, (size_t)Nt)) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc gap", e);
  if ((e = cudaMalloc((void**)&ctx->vprefix, ((size_t)Nt + 1) * sizeof(int))) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc vprefix", e);
  if ((e = cudaMalloc((void**)&ctx->valid_m, (size_t)ncol_cap * sizeof(int))) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc valid_m", e);
  if ((e = cudaMalloc((void**)&ctx->lut, (kLutN + 1) * sizeof(float4))) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc lut", e);
  if ((e = cudaMalloc((void**)&ctx->bad, sizeof(unsigned long long))) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc counter", e);
  if ((e = cudaMalloc((void**)&ctx->work, 2 * sizeof(unsigned long long))) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc counter", e);
  if ((e = cudaMalloc((void**)&ctx->census, 5 * sizeof(unsigned long long))) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc counter", e);
  if ((e = cudaMemset(ctx->census, 0, 5 * sizeof(unsigned long long))) != cudaSuccess) return bail(TFS_ECUDA, "cudaMemset counter", e);
  if ((e = cudaFuncSetAttribute(eval_list_kernel<0, kWGeneral>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_list_kernel<0, kWSeparable>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_list_kernel<0, kWTimeOnly>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_list_kernel<1, kWGeneral>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_list_kernel<2, kWGeneral>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_list_kernel<2, kWSeparable>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_list_kernel<2, kWTimeOnly>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_wdm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_slab_kernel<kWGeneral>, cudaFuncAttributeMaxDynamicSharedMemorySize, slab_smem_bytes(kWGeneral))) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_slab_kernel<kWSeparable>, cudaFuncAttributeMaxDynamicSharedMemorySize, slab_smem_bytes(kWSeparable))) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_slab_kernel<kWTimeOnly>, cudaFuncAttributeMaxDynamicSharedMemorySize, slab_smem_bytes(kWTimeOnly))) != cudaSuccess ||
      // the counting builds of tfs_tier_census
      (e = cudaFuncSetAttribute(eval_list_kernel<0, kWGeneral, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_list_kernel<0, kWSeparable, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_list_kernel<0, kWTimeOnly, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kLutListBytes)) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_slab_kernel<kWGeneral, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, slab_smem_bytes(kWGeneral))) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_slab_kernel<kWSeparable, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, slab_smem_bytes(kWSeparable))) != cudaSuccess ||
      (e = cudaFuncSetAttribute(eval_slab_kernel<kWTimeOnly, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, slab_smem_bytes(kWTimeOnly))) != cudaSuccess)
    return bail(TFS_ECUDA, "cudaFuncSetAttribute(max dynamic shared memory)", e);
  if ((e = cudaMalloc((void**)&ctx->sel, sizeof(SelectState))) != cudaSuccess) return bail(TFS_ENOMEM, "cudaMalloc select state", e);
  std::vector<float4> lut;
  build_lut(lut);
  if (!(fit_far(ctx->far) < 2e-6)) return bail(TFS_ECUDA, "far-zone polynomial fit failed", cudaSuccess);
  if ((e = cudaMemcpy(ctx->lut, lut.data(), lut.size() * sizeof(float4), cudaMemcpyHostToDevice)) != cudaSuccess)
    return bail(TFS_ECUDA, "cudaMemcpy lut", e);
  *out = ctx;
  return TFS_OK;
}

int tfs_set_profiling(tfs_ctx* ctx, int on) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_set_profiling: ctx is NULL");
  ctx->profiling = (on != 0);
  ctx->ev_used = 0;
  ctx->launches = 0;
  return TFS_OK;
}

int tfs_tier_census(tfs_ctx* ctx, int on, long long* counts) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_tier_census: ctx is NULL");
  int rc = check_device(ctx, "tfs_tier_census");
  if (rc) return rc;
  TFS_CUDA(ctx, cudaDeviceSynchronize());
  if (counts) {
    unsigned long long h[5];
    TFS_CUDA(ctx, cudaMemcpy(h, ctx->census, sizeof(h), cudaMemcpyDeviceToHost));
    for (int i = 0; i < 5; ++i) counts[i] = (long long)h[i];
  }
  TFS_CUDA(ctx, cudaMemset(ctx->census, 0, 5 * sizeof(unsigned long long)));
  ctx->census_on = (on != 0);
  return TFS_OK;
}

int tfs_get_profile_kernels(tfs_ctx* ctx, double* slab_kernel_ms, double* list_kernel_ms, long long* eval_launches,
                            long long* kernel_launches) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_get_profile_kernels: ctx is NULL");
  double ms_list = 0.0, ms_slab = 0.0;
  for (size_t i = 0; i + 3 <= ctx->ev_used; i += 3) {
    float t = 0.f;
    TFS_CUDA(ctx, cudaEventSynchronize(ctx->ev_pool[i + 2]));
    TFS_CUDA(ctx, cudaEventElapsedTime(&t, ctx->ev_pool[i], ctx->ev_pool[i + 1]));
    ms_list += t;
    TFS_CUDA(ctx, cudaEventElapsedTime(&t, ctx->ev_pool[i + 1], ctx->ev_pool[i + 2]));
    ms_slab += t;
  }
  if (slab_kernel_ms) *slab_kernel_ms = ms_slab;
  if (list_kernel_ms) *list_kernel_ms = ms_list;
  if (eval_launches) *eval_launches = (long long)(ctx->ev_used / 3);
  if (kernel_launches) *kernel_launches = ctx->launches;
  return TFS_OK;
}

int tfs_get_profile(tfs_ctx* ctx, double* main_kernel_ms, long long* main_kernel_launches, long long* kernel_launches) {
  double a = 0.0, b = 0.0;
  const int rc = tfs_get_profile_kernels(ctx, &a, &b, main_kernel_launches, kernel_launches);
  if (rc == TFS_OK && main_kernel_ms) *main_kernel_ms = a + b;
  return rc;
}

void tfs_destroy(tfs_ctx* ctx) {
  if (!ctx) return;
  if (ctx->l2_window_used)
    fprintf(stderr, "tfs: TFS_L2_WINDOW=1: %lld evaluation launches ran with the grid declared persisting in L2\n", ctx->l2_window_used);
  for (auto& ev : ctx->ev_pool) cudaEventDestroy(ev);
  void* bufs[] = {ctx->pair[0].grid, ctx->pair[0].wgt, ctx->pair[0].wa, ctx->pair[0].wb, ctx->pair[1].grid, ctx->pair[1].wgt,
                  ctx->pair[1].wa, ctx->pair[1].wb, ctx->colmax, ctx->wcounts, ctx->gap, ctx->vprefix, ctx->valid_m, ctx->lut,
                  ctx->bad, ctx->work, ctx->census, ctx->sel, ctx->buf_params, ctx->buf_partials, ctx->buf_prep, ctx->buf_ttab,
                  ctx->buf_out[0], ctx->buf_out[1], ctx->buf_out[2], ctx->buf_out[3], ctx->buf_out[4], ctx->buf_keys,
                  ctx->buf_tk_in, ctx->buf_tk_idx, ctx->buf_tk_val, ctx->buf_counts, ctx->buf_children, ctx->buf_fe};
  for (void* b : bufs) if (b) cudaFree(b);
  free_piece_tables(ctx);
  delete ctx;
}

// The upload proper.  sep_bk: the caller KNOWS the weights are W[a,m,k] = bk[a][k] (device table [C][Nf], or NULL for
// W = 1) and passes weight == NULL: no per-pixel weight array is written, read or analysed (the time-series front end).
static int upload_impl(tfs_ctx* ctx, const float* coeff, const float* weight, const uint8_t* gap_mask, void* stream,
                       bool sep_known, const float* sep_bk) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_upload_data: ctx is NULL");
  if (!coeff) return fail(ctx, TFS_EINVAL, "tfs_upload_data: coeff is NULL");
  int rc = check_device(ctx, "tfs_upload_data");
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t npix = (size_t)ctx->Nt * ctx->Nf;
  const int C = ctx->C;
  const float* d_coeff = coeff;
  const float* d_weight = weight;
  void* tmp_c = nullptr;
  void* tmp_w = nullptr;
  auto cleanup = [&]() { if (tmp_c) cudaFree(tmp_c); if (tmp_w) cudaFree(tmp_w); };
#define UP_CUDA(expr)                                                                      \
  do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { cleanup();                       \
       return fail(ctx, e_ == cudaErrorMemoryAllocation ? TFS_ENOMEM : TFS_ECUDA,          \
                   "%s failed: %s", #expr, cudaGetErrorString(e_)); } } while (0)
  const size_t cfl = ctx->opts.basis == 1 ? 1 : 2;          // floats per coefficient: real WDM pixels / complex tranche bins
  if (!is_device_ptr(coeff)) {
    UP_CUDA(cudaMalloc(&tmp_c, npix * C * cfl * sizeof(float)));
    UP_CUDA(cudaMemcpyAsync(tmp_c, coeff, npix * C * cfl * sizeof(float), cudaMemcpyHostToDevice, st));
    d_coeff = (const float*)tmp_c;
  }
  if (weight && !is_device_ptr(weight)) {
    UP_CUDA(cudaMalloc(&tmp_w, npix * C * sizeof(float)));
    UP_CUDA(cudaMemcpyAsync(tmp_w, weight, npix * C * sizeof(float), cudaMemcpyHostToDevice, st));
    d_weight = (const float*)tmp_w;
  }
  if (gap_mask) {
    UP_CUDA(cudaMemcpyAsync(ctx->gap, gap_mask, (size_t)ctx->Nt,
                            is_device_ptr(gap_mask) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
  } else {
    UP_CUDA(cudaMemsetAsync(ctx->gap, 1, (size_t)ctx->Nt, st));
  }
  // the compacted list of valid tranches comes first: the grid is stored over it (gap tranches are not kept)
  valid_list_kernel<<<1, 1024, 0, st>>>(ctx->gap, ctx->Nt, ctx->ncol_cap, ctx->vprefix, ctx->valid_m);
  UP_CUDA(cudaGetLastError());
  int n_valid = 0;
  UP_CUDA(cudaMemcpyAsync(&n_valid, ctx->vprefix + ctx->Nt, sizeof(int), cudaMemcpyDeviceToHost, st));
  UP_CUDA(cudaStreamSynchronize(st));
  ctx->n_valid = n_valid;
  ctx->ncol = std::max(1, (n_valid + kTS - 1) / kTS) * kTS;
  free_piece_tables(ctx);                  // cut for the previous gap mask
  const size_t nrow = (size_t)ctx->Nf + kPadRows;
  const dim3 blocks((unsigned)((ctx->Nf + 31) / 32), (unsigned)((ctx->Nt + 31) / 32));
  if (ctx->opts.basis == 1) {
    // WDM pixels: real coefficients [C][Nt][Nf]; y = W d and W as float2 planes in the pair's buffers
    tfs_ctx::Pair& P = ctx->pair[0];
    UP_CUDA(cudaMemsetAsync(P.grid, 0, nrow * ctx->ncol * sizeof(float2), st));
    UP_CUDA(cudaMemsetAsync(P.wgt, 0, nrow * ctx->ncol * sizeof(float2), st));
    pack_wdm_kernel<<<blocks, 256, 0, st>>>(d_coeff, d_weight, ctx->Nt, ctx->Nf, C, ctx->gap, ctx->vprefix, ctx->ncol,
                                            (float2*)P.grid, P.wgt);
    UP_CUDA(cudaGetLastError());
    ctx->launches += 2;
    UP_CUDA(cudaStreamSynchronize(st));
    ctx->wmode = kWGeneral;
    cleanup();
    ctx->uploaded = true;
    return TFS_OK;
  }
  int wmode = kWTimeOnly;
  for (int pr = 0; pr < ctx->n_pairs; ++pr) {
    tfs_ctx::Pair& P = ctx->pair[pr];
    UP_CUDA(cudaMemsetAsync(P.grid, 0, nrow * ctx->ncol * sizeof(float4), st));
    if (!sep_known) UP_CUDA(cudaMemsetAsync(P.wgt, 0, nrow * ctx->ncol * sizeof(float2), st));
    pack_kernel<<<blocks, 256, 0, st>>>((const float2*)d_coeff, d_weight, sep_known ? sep_bk : nullptr, ctx->Nt, ctx->Nf, P.c0,
                                        P.c1, ctx->gap, ctx->vprefix, ctx->ncol, P.grid, sep_known ? nullptr : P.wgt);
    UP_CUDA(cudaGetLastError());
    ctx->launches += 1;
    // weight structure (C11): W = a[i] b[k] on every pixel?  then the hot loop reads no per-pixel weight
    unsigned long long wc[2] = {1, 1};
    if (sep_known) {
      UP_CUDA(cudaMemsetAsync(ctx->wcounts, 0, 2 * sizeof(unsigned long long), st));
      UP_CUDA(cudaMemsetAsync(P.wa, 0, (size_t)ctx->ncol_cap * sizeof(float2), st));
      weight_sep_set_kernel<<<1, 1024, 0, st>>>(sep_bk, ctx->Nf, P.c0, P.c1, n_valid, P.wa, P.wb, ctx->wcounts);
      UP_CUDA(cudaGetLastError());
      ctx->launches += 1;
      UP_CUDA(cudaMemcpyAsync(wc, ctx->wcounts, sizeof(wc), cudaMemcpyDeviceToHost, st));
      UP_CUDA(cudaStreamSynchronize(st));
    } else if (ctx->opts.weight_mode == 0) {
      UP_CUDA(cudaMemsetAsync(ctx->wcounts, 0, 2 * sizeof(unsigned long long), st));
      weight_colmax_kernel<<<(unsigned)ctx->Nf, 256, 0, st>>>(P.wgt, ctx->ncol, n_valid, ctx->colmax);
      UP_CUDA(cudaMemsetAsync(P.wa, 0, (size_t)ctx->ncol_cap * sizeof(float2), st));
      weight_rowmax_kernel<<<dim3((unsigned)((std::max(n_valid, 1) + 127) / 128), 32), 128, 0, st>>>(P.wgt, ctx->ncol, n_valid, ctx->Nf, P.wa);
      weight_factor_kernel<<<1, 1024, 0, st>>>(ctx->colmax, ctx->Nf, P.wb, ctx->wcounts);
      weight_check_kernel<<<(unsigned)(((size_t)ctx->ncol * ctx->Nf + 255) / 256), 256, 0, st>>>(P.wgt, P.wa, P.wb, ctx->ncol, n_valid,
                                                                                              ctx->Nf, ctx->wcounts);
      UP_CUDA(cudaGetLastError());
      ctx->launches += 4;
      UP_CUDA(cudaMemcpyAsync(wc, ctx->wcounts, sizeof(wc), cudaMemcpyDeviceToHost, st));
      UP_CUDA(cudaStreamSynchronize(st));
    }
    const int wm = wc[0] != 0 ? kWGeneral : (wc[1] != 0 ? kWSeparable : kWTimeOnly);
    wmode = std::min(wmode, wm);           // the most general structure among the pairs decides the kernel
  }
  ctx->launches += 1;
  UP_CUDA(cudaStreamSynchronize(st));
  ctx->wmode = wmode;
  cleanup();
#undef UP_CUDA
  // TMA descriptors of the slab kernel (the box height depends on the weight structure)
  for (int pr = 0; pr < ctx->n_pairs; ++pr) {
    tfs_ctx::Pair& P = ctx->pair[pr];
    rc = encode_map(ctx, &P.map_y, P.grid, 4, ctx->ncol, (int)nrow, slab_rows(wmode));
    if (rc) return rc;
    rc = encode_map(ctx, &P.map_w, P.wgt, 2, ctx->ncol, (int)nrow, slab_rows(wmode));
    if (rc) return rc;
  }
  ctx->uploaded = true;
  return TFS_OK;
}

int tfs_upload_data(tfs_ctx* ctx, const float* coeff, const float* weight, const uint8_t* gap_mask, void* stream) {
  return upload_impl(ctx, coeff, weight, gap_mask, stream, false, nullptr);
}

int tfs_upload_timeseries(tfs_ctx* ctx, const float* x, const uint8_t* sample_mask, const float* psd,
                          double tukey_alpha, float* coeff_out, float* weight_out, uint8_t* gap_out, void* stream) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_upload_timeseries: ctx is NULL");
  if (!x) return fail(ctx, TFS_EINVAL, "tfs_upload_timeseries: x is NULL");
  if (!(tukey_alpha >= 0.0 && tukey_alpha <= 1.0))
    return fail(ctx, TFS_EINVAL, "tfs_upload_timeseries: tukey_alpha must be in [0, 1] (got %g)", tukey_alpha);
  if (int rcd = check_device(ctx, "tfs_upload_timeseries")) return rcd;
  if (ctx->opts.basis != 0) return fail(ctx, TFS_EINVAL, "tfs_upload_timeseries: the front end builds short-time Fourier tranches (basis 0)");
  if (ctx->Nt > 65535) return fail(ctx, TFS_EINVAL, "tfs_upload_timeseries: Nt must be <= 65535 (got %d)", ctx->Nt);
  cudaStream_t st = (cudaStream_t)stream;
  const int C = ctx->C, Nt = ctx->Nt, Nf = ctx->Nf, N = 2 * ctx->Nf;
  // radices of the length-Nf complex FFT behind the packed real transform
  FeRadices rad{};
  {
    int L = Nf;
    const int primes[4] = {4, 2, 3, 5};
    for (int pi = 0; pi < 4; ++pi)
      while (L % primes[pi] == 0 && rad.n < kFeMaxStages) { rad.r[rad.n++] = primes[pi]; L /= primes[pi]; }
    if (L != 1) return fail(ctx, TFS_EINVAL, "tfs_upload_timeseries: Nf = %d must factor into 2, 3 and 5", Nf);
    int Ns = 1;
    for (int s = 0; s < rad.n; ++s) { rad.off[s] = rad.total; rad.total += (rad.r[s] - 1) * Ns; Ns *= rad.r[s]; }
  }
  const size_t smem = 2 * (size_t)Nf * sizeof(float2);
  if (smem > 200 * 1024) return fail(ctx, TFS_EINVAL, "tfs_upload_timeseries: Nf = %d is too long for the shared-memory FFT", Nf);
  const size_t nsamp = (size_t)Nt * N, npix = (size_t)Nt * Nf;
  // one pooled scratch allocation, kept in the context (a second dataset of the same size costs no cudaMalloc)
  const bool copy_x = !is_device_ptr(x) || ((uintptr_t)x & 7u);
  const bool copy_mask = sample_mask && !is_device_ptr(sample_mask);
  const bool copy_psd = psd && !is_device_ptr(psd);
  auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
  // the per-pixel weight array is only materialised when the caller wants it back or forces the general path:
  // W[a,m,k] = b_a[k] is separable by construction, so the upload takes the table b directly
  // (fresnel_mode 1 always evaluates with the general-weight kernel, which reads the per-pixel array: it needs it too)
  const bool per_pixel_w = ctx->opts.weight_mode != 0 || ctx->opts.fresnel_mode != 0;
  const bool need_w = weight_out != nullptr || per_pixel_w;
  const size_t sz[7] = {copy_x ? al(C * nsamp * sizeof(float)) : 0, copy_mask ? al(nsamp) : 0,
                        copy_psd ? al((size_t)C * Nf * sizeof(float)) : 0, al((size_t)(rad.total + 2) * sizeof(float2)),
                        al((size_t)N * sizeof(float)), al(C * npix * sizeof(float2)), need_w ? al(C * npix * sizeof(float)) : 0};
  size_t total = al((size_t)Nt) + al((size_t)C * Nf * sizeof(float));
  for (size_t b : sz) total += b;
  int rc0 = ensure(ctx, &ctx->buf_fe, &ctx->cap_fe, total);
  if (rc0) return rc0;
  char* base = (char*)ctx->buf_fe;
  char* part[8];
  for (int i = 0; i < 7; ++i) { part[i] = base; base += sz[i]; }
  part[7] = base;
#define FE_CUDA(expr) TFS_CUDA(ctx, expr)
  const float* d_x = x;
  if (copy_x) {
    FE_CUDA(cudaMemcpyAsync(part[0], x, C * nsamp * sizeof(float), cudaMemcpyDefault, st));
    d_x = (const float*)part[0];
  }
  const uint8_t* d_mask = sample_mask;
  if (copy_mask) {
    FE_CUDA(cudaMemcpyAsync(part[1], sample_mask, nsamp, cudaMemcpyHostToDevice, st));
    d_mask = (const uint8_t*)part[1];
  }
  const float* d_psd = psd;
  if (copy_psd) {
    FE_CUDA(cudaMemcpyAsync(part[2], psd, (size_t)C * Nf * sizeof(float), cudaMemcpyHostToDevice, st));
    d_psd = (const float*)part[2];
  }
  float2* d_tw = (float2*)part[3];
  float* d_win = (float*)part[4];
  float2* d_coeff = (float2*)part[5];
  float* d_weight = (float*)part[6];
  uint8_t* d_gap = (uint8_t*)part[7];
  float* d_bk = (float*)(part[7] + al((size_t)Nt));

  fe_tables_kernel<<<(unsigned)((std::max(N, rad.total) + 255) / 256), 256, 0, st>>>(d_tw, rad, d_win, N, tukey_alpha);
  FE_CUDA(cudaGetLastError());
  FE_CUDA(cudaFuncSetAttribute(fe_fft_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  fe_gap_kernel<<<(unsigned)Nt, 256, 0, st>>>(d_mask, N, d_gap);          // before the FFT: it also clears g[m] on non-finite samples
  FE_CUDA(cudaGetLastError());
  fe_fft_kernel<<<dim3((unsigned)Nt, (unsigned)C), kFeThreads, smem, st>>>(d_x, d_win, d_tw, rad, Nt, Nf, d_coeff, d_gap);
  FE_CUDA(cudaGetLastError());
  ctx->launches += 3;
  if (need_w) {
    fe_weight_kernel<<<dim3((unsigned)((Nf + 255) / 256), (unsigned)Nt, (unsigned)C), 256, 0, st>>>(d_psd, Nt, Nf, ctx->DT, d_weight);
    FE_CUDA(cudaGetLastError());
    ctx->launches += 1;
  }
  if (d_psd) {
    fe_bk_kernel<<<(unsigned)((C * Nf + 255) / 256), 256, 0, st>>>(d_psd, C, Nf, ctx->DT, d_bk);
    FE_CUDA(cudaGetLastError());
    ctx->launches += 1;
  }
  if (coeff_out) FE_CUDA(cudaMemcpyAsync(coeff_out, d_coeff, C * npix * sizeof(float2), cudaMemcpyDefault, st));
  if (weight_out) FE_CUDA(cudaMemcpyAsync(weight_out, d_weight, C * npix * sizeof(float), cudaMemcpyDefault, st));
  if (gap_out) FE_CUDA(cudaMemcpyAsync(gap_out, d_gap, (size_t)Nt, cudaMemcpyDefault, st));
#undef FE_CUDA
  // the rest is the ordinary upload, from device buffers (it synchronises the stream before returning); with the
  // default weight_mode the weights go in as the per-bin table (no per-pixel array is read or analysed)
  if (per_pixel_w) return upload_impl(ctx, (const float*)d_coeff, d_weight, d_gap, stream, false, nullptr);
  return upload_impl(ctx, (const float*)d_coeff, nullptr, d_gap, stream, true, d_psd ? d_bk : nullptr);
}

}  // extern "C"

namespace {

template <int WMODE>
void launch_slab(const EvalArgs& a, const tfs_ctx::Pair& P, unsigned blocks, cudaStream_t st) {
  if (a.census) eval_slab_kernel<WMODE, true><<<blocks, kSlabWarps * 32, slab_smem_bytes(WMODE), st>>>(a, P.map_y, P.map_w);
  else eval_slab_kernel<WMODE><<<blocks, kSlabWarps * 32, slab_smem_bytes(WMODE), st>>>(a, P.map_y, P.map_w);
}

// the list kernel of the default template (MODE 0): the counting build while a tier census is on
template <int WMODE>
void launch_list0(const EvalArgs& a, unsigned blocks, cudaStream_t st) {
  if (a.census) eval_list_kernel<0, WMODE, true><<<blocks, kWarpsPerCta * 32, kLutListBytes, st>>>(a);
  else eval_list_kernel<0, WMODE><<<blocks, kWarpsPerCta * 32, kLutListBytes, st>>>(a);
}

// the evaluation proper (rows a1-a8) for one batch; `transfer` = per-template table [n][C][n_knots] complex or NULL
int eval_impl(tfs_ctx* ctx, const double* params, long long n, int N_seg, const float* transfer, int n_knots,
              double f_knot0, double f_knot_step, float* upsilon, float* seg_power, float* seg_dh, float* seg_hh,
              void* stream, const char* who, int M_tr = 0, int* n_seg_eff = nullptr) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "%s: ctx is NULL", who);
  if (n < 0) return fail(ctx, TFS_EINVAL, "%s: n < 0", who);
  if (M_tr < 0) return fail(ctx, TFS_EINVAL, "%s: seg_tranches must be >= 1", who);
  if (M_tr > 0) N_seg = (ctx->Nt + M_tr - 1) / M_tr;
  if (n_seg_eff && ctx->opts.basis == 1) return fail(ctx, TFS_EINVAL, "%s: n_seg_eff is not available in the WDM basis", who);
  if (N_seg < 1 || N_seg > ctx->Nt) return fail(ctx, TFS_EINVAL, "%s: need 1 <= N_seg <= Nt (got %d, Nt %d)", who, N_seg, ctx->Nt);
  if (!ctx->uploaded) return fail(ctx, TFS_ESTATE, "%s: no data uploaded (call tfs_upload_data first)", who);
  if (transfer && ctx->opts.basis == 1) return fail(ctx, TFS_EINVAL, "%s: transfer tables are not available in the WDM basis", who);
  if (transfer && (n_knots < 1 || n_knots > 65536 || !std::isfinite(f_knot0) || (n_knots > 1 && !(f_knot_step > 0.0))))
    return fail(ctx, TFS_EINVAL, "%s: transfer table needs 1 <= n_knots <= 65536, finite f_knot0 and f_knot_step > 0", who);
  if (ctx->C == 3 && !transfer && !ctx->t3_set)
    return fail(ctx, TFS_EINVAL, "%s: the parameter row has no column for the third channel's transfer factor: declare it with "
                                 "tfs_set_third_channel_factor (0, 0 drops the channel) or pass a table to tfs_eval_tf", who);
  int rc = check_device(ctx, who);
  if (rc) return rc;
  if (n == 0) { ctx->bad_host = 0; return TFS_OK; }
  if (!params || !upsilon) return fail(ctx, TFS_EINVAL, "%s: params and upsilon are required", who);
  if (n >= (1ll << 32)) return fail(ctx, TFS_EINVAL, "%s: n must be < 2^32", who);
  cudaStream_t st = (cudaStream_t)stream;
  const int C = ctx->C;

  const double* d_params = nullptr;
  rc = stage_params(ctx, params, n, st, &d_params);
  if (rc) return rc;
  const float2* d_ttab = (const float2*)transfer;
  if (transfer && !is_device_ptr(transfer)) {
    const size_t bytes = (size_t)n * C * n_knots * sizeof(float2);
    rc = ensure(ctx, &ctx->buf_ttab, &ctx->cap_ttab, bytes);
    if (rc) return rc;
    TFS_CUDA(ctx, cudaMemcpyAsync(ctx->buf_ttab, transfer, bytes, cudaMemcpyHostToDevice, st));
    d_ttab = (const float2*)ctx->buf_ttab;
  }

  // outputs: device pointers are written in place, host pointers via ctx scratch + D2H
  float* user[5] = {upsilon, seg_power, seg_dh, seg_hh, reinterpret_cast<float*>(n_seg_eff)};   // int32 rides as 4-byte words
  const size_t per[5] = {1, (size_t)N_seg, (size_t)N_seg * 2, (size_t)N_seg, 1};
  float* dev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  bool host_out[5] = {false, false, false, false, false};
  bool any_host = false;
  for (int i = 0; i < 5; ++i) {
    if (!user[i]) continue;
    if (is_device_ptr(user[i])) { dev[i] = user[i]; continue; }
    host_out[i] = true; any_host = true;
    rc = ensure(ctx, &ctx->buf_out[i], &ctx->cap_out[i], (size_t)n * per[i] * sizeof(float));
    if (rc) return rc;
    dev[i] = (float*)ctx->buf_out[i];
  }

  // tiling: tiles of kTS valid tranches, cut by the segment boundaries into pieces (one partial each)
  const tfs_ctx::PieceTable* pt = nullptr;
  rc = get_piece_table(ctx, N_seg, M_tr, st, &pt);
  if (rc) return rc;
  const int n_tiles = pt->n_tiles;
  const size_t max_pieces = (size_t)n_tiles + (size_t)N_seg;
  const bool wdm = ctx->opts.basis == 1;
  const size_t part_bytes = (wdm ? 2 : 1) * sizeof(float4);          // per (piece, template)
  long long sub = (long long)(kScratchBytes / (max_pieces * part_bytes));
  sub = std::max<long long>(sub, 1024);
  sub = std::min<long long>(sub, n);
  rc = ensure(ctx, &ctx->buf_partials, &ctx->cap_partials, (size_t)sub * max_pieces * part_bytes);
  if (rc) return rc;

  // pre-pass scratch (one pooled allocation): constants, keys, bucket tables, item list, unit tables
  const int n_bands = (ctx->Nf - 1) / kBandStride + 1;
  const bool windowed = ctx->opts.tukey_alpha > 0.0;          // window-aware template: every item through the list kernel (MODE 2)
  const bool slab_ok = ctx->opts.fresnel_mode == 0 && n_bands + 2 <= 8192 && !wdm && !windowed;
  const int n_keys = slab_ok ? n_bands + 2 : 2;
  const size_t n_buckets = (size_t)n_tiles * n_keys;
  const size_t n_items = (size_t)sub * n_tiles;
  const size_t max_us = n_items / kUnitItems + n_buckets + 1, max_ul = n_items / kListUnitItems + (size_t)n_tiles + 1;
  auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
  const size_t sz[8] = {al((size_t)sub * sizeof(TplConst)), al(n_items * sizeof(uint16_t)), al(n_buckets * sizeof(unsigned)),
                        al(n_buckets * sizeof(unsigned)), al(n_items * sizeof(unsigned)), al(max_us * sizeof(Unit)),
                        al(max_ul * sizeof(Unit)), al(2 * sizeof(int))};
  size_t total = 0;
  for (size_t b : sz) total += b;
  rc = ensure(ctx, &ctx->buf_prep, &ctx->cap_prep, total);
  if (rc) return rc;
  char* part[8];
  { char* q = (char*)ctx->buf_prep; for (int i = 0; i < 8; ++i) { part[i] = q; q += sz[i]; } }
#ifdef TFS_POISON
  // debug builds only (the initcheck substitute, tests/test_gpu_parity.py): every scratch buffer starts as NaN /
  // 0xFFFF... patterns, so a value read before it was written shows up in the outputs
  TFS_CUDA(ctx, cudaMemsetAsync(ctx->buf_partials, 0xFF, (size_t)sub * max_pieces * part_bytes, st));
  TFS_CUDA(ctx, cudaMemsetAsync(ctx->buf_prep, 0xFF, total, st));
  for (int i = 0; i < 5; ++i)
    if (host_out[i]) TFS_CUDA(ctx, cudaMemsetAsync(dev[i], 0xFF, (size_t)n * per[i] * sizeof(float), st));
#endif

  TFS_CUDA(ctx, cudaMemsetAsync(ctx->bad, 0, sizeof(unsigned long long), st));
  const int wm = ctx->opts.fresnel_mode != 0 ? kWGeneral : ctx->wmode;
  // channel pairs to run: the pair of channel 2 only when it has a transfer factor -- from the table, or the context's
  // constant T_T when that is not zero
  const bool t3_const = !d_ttab && (ctx->t3[0] != 0.0 || ctx->t3[1] != 0.0);
  const int n_pass = (ctx->n_pairs == 2 && (d_ttab || t3_const)) ? 2 : 1;
  for (long long off = 0; off < n; off += sub) {
    const long long nb = std::min(sub, n - off);
    for (int pass = 0; pass < n_pass; ++pass) {
      EvalArgs a = base_args(ctx, pass);
      a.n_tiles = n_tiles; a.n_keys = n_keys; a.slab_ok = slab_ok ? 1 : 0; a.wmode = wm;
      a.tile_first = pt->tile_first;
      a.piece_end = pt->piece_end;
      a.partials = (float4*)ctx->buf_partials;
      a.params = d_params + off * TFS_PARAM_COLS;
      a.n = nb;
      a.tconst = (TplConst*)part[0]; a.keys = (uint16_t*)part[1]; a.counts = (unsigned*)part[2];
      a.bucket_off = (unsigned*)part[3]; a.list = (unsigned*)part[4]; a.units_slab = (Unit*)part[5];
      a.units_list = (Unit*)part[6]; a.n_units = (int*)part[7];
      a.accumulate = pass;
      a.t_col = pass == 0 ? 3 : -1;
      a.t3_re = ctx->t3[0]; a.t3_im = ctx->t3[1];
      if (pass > 0) a.bad_count = nullptr;
      if (d_ttab) {
        a.ttab = d_ttab + (size_t)off * C * n_knots;
        a.tt_K = n_knots; a.tt_C = C; a.tt_ch0 = ctx->pair[pass].c0;
        const double step = n_knots > 1 ? f_knot_step : 1.0;
        a.tt_scale = (float)(1.0 / (ctx->DT * step));        // knot position of bin x: (x/DT - f0)/step
        a.tt_off = (float)(f_knot0 / step);
      }
      const unsigned tb = (unsigned)((nb + 255) / 256);
      prep_consts_kernel<<<tb, 256, 0, st>>>(a);
      ctx->launches += 1;
      if (pass == 0) {
        TFS_CUDA(ctx, cudaMemsetAsync(a.counts, 0, n_buckets * sizeof(unsigned), st));
        const unsigned tbp = (unsigned)((nb + 256 * kPrepItems - 1) / (256 * kPrepItems));
        prep_keys_kernel<<<dim3(tbp, (unsigned)n_tiles), 256, n_keys * sizeof(unsigned), st>>>(a);
        prep_scan_kernel<<<1, 1024, 0, st>>>(a);
        prep_scatter_kernel<<<dim3(tbp, (unsigned)n_tiles), 256, 2 * n_keys * sizeof(unsigned), st>>>(a);
        ctx->launches += 3;
      }
      TFS_CUDA(ctx, cudaGetLastError());
      TFS_CUDA(ctx, cudaMemsetAsync(ctx->work, 0, 2 * sizeof(unsigned long long), st));
      cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
      if (ctx->profiling) {
        while (ctx->ev_pool.size() < ctx->ev_used + 3) {
          cudaEvent_t e0;
          TFS_CUDA(ctx, cudaEventCreate(&e0));
          ctx->ev_pool.push_back(e0);
        }
        for (int i = 0; i < 3; ++i) ev[i] = ctx->ev_pool[ctx->ev_used + i];
        ctx->ev_used += 3;
        TFS_CUDA(ctx, cudaEventRecord(ev[0], st));
      }
      const unsigned blocks = (unsigned)ctx->sm_count;       // persistent, 1 CTA per SM
      // Measurement aid (BASELINE.json north_star (2): "the grid pinned in L2 through an access-policy window when it
      // fits"): with TFS_L2_WINDOW=1 in the environment the pair's grid is declared persisting for the two evaluation
      // launches when it fits the device's persisting-L2 limit.  Off by default: DESIGN.md section 7 has the measurement.
      bool l2win = false;
      {
        static const bool want = [] { const char* e = getenv("TFS_L2_WINDOW"); return e && e[0] == '1'; }();
        const size_t gbytes = ((size_t)ctx->Nf + kPadRows) * ctx->ncol * sizeof(float4);
        int max_persist = 0, max_win = 0;
        if (want && cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, ctx->device) == cudaSuccess &&
            cudaDeviceGetAttribute(&max_win, cudaDevAttrMaxAccessPolicyWindowSize, ctx->device) == cudaSuccess &&
            gbytes <= (size_t)max_persist && gbytes <= (size_t)max_win) {
          cudaStreamAttrValue v{};
          v.accessPolicyWindow.base_ptr = (void*)ctx->pair[pass].grid;
          v.accessPolicyWindow.num_bytes = gbytes;
          v.accessPolicyWindow.hitRatio = 1.0f;
          v.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
          v.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
          l2win = cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, gbytes) == cudaSuccess &&
                  cudaStreamSetAttribute(st, cudaStreamAttributeAccessPolicyWindow, &v) == cudaSuccess;
          cudaGetLastError();
          ctx->l2_window_used += l2win ? 1 : 0;
        }
      }
      // the items that gather from global memory (and every item with the paper's approximants) ...
      if (wdm) eval_wdm_kernel<<<blocks, kWarpsPerCta * 32, kLutListBytes, st>>>(a);
      else if (ctx->opts.fresnel_mode != 0) eval_list_kernel<1, kWGeneral><<<blocks, kWarpsPerCta * 32, kLutListBytes, st>>>(a);
      else if (windowed && wm == kWTimeOnly) eval_list_kernel<2, kWTimeOnly><<<blocks, kWarpsPerCta * 32, kLutListBytes, st>>>(a);
      else if (windowed && wm == kWSeparable) eval_list_kernel<2, kWSeparable><<<blocks, kWarpsPerCta * 32, kLutListBytes, st>>>(a);
      else if (windowed) eval_list_kernel<2, kWGeneral><<<blocks, kWarpsPerCta * 32, kLutListBytes, st>>>(a);
      else if (wm == kWTimeOnly) launch_list0<kWTimeOnly>(a, blocks, st);
      else if (wm == kWSeparable) launch_list0<kWSeparable>(a, blocks, st);
      else launch_list0<kWGeneral>(a, blocks, st);
      TFS_CUDA(ctx, cudaGetLastError());
      if (ev[1]) TFS_CUDA(ctx, cudaEventRecord(ev[1], st));
      ctx->launches += 1;
      // ... and the band buckets from shared-memory slabs
      if (slab_ok) {
        if (wm == kWTimeOnly) launch_slab<kWTimeOnly>(a, ctx->pair[pass], blocks, st);
        else if (wm == kWSeparable) launch_slab<kWSeparable>(a, ctx->pair[pass], blocks, st);
        else launch_slab<kWGeneral>(a, ctx->pair[pass], blocks, st);
        TFS_CUDA(ctx, cudaGetLastError());
        ctx->launches += 1;
      }
      if (ev[2]) TFS_CUDA(ctx, cudaEventRecord(ev[2], st));
      if (l2win) {
        cudaStreamAttrValue v{};
        v.accessPolicyWindow.num_bytes = 0;
        cudaStreamSetAttribute(st, cudaStreamAttributeAccessPolicyWindow, &v);
        cudaGetLastError();
      }
    }
    const int threads = 128;
    if (wdm)
      combine_wdm_kernel<<<(unsigned)((nb + threads - 1) / threads), threads, 0, st>>>(
          (const float4*)ctx->buf_partials, (const uint16_t*)part[1], nb, N_seg, pt->tile_first, n_tiles, pt->piece_seg,
          pt->piece_tile, dev[0] + off, dev[1] ? dev[1] + off * per[1] : nullptr,
          dev[2] ? dev[2] + off * per[2] : nullptr, dev[3] ? dev[3] + off * per[3] : nullptr);
    else
    combine_kernel<<<(unsigned)((nb + threads - 1) / threads), threads, 0, st>>>(
        (const float4*)ctx->buf_partials, (const uint16_t*)part[1], nb, N_seg, pt->tile_first, n_tiles, pt->piece_seg,
        pt->piece_tile, dev[0] + off, dev[1] ? dev[1] + off * per[1] : nullptr,
        dev[2] ? dev[2] + off * per[2] : nullptr, dev[3] ? dev[3] + off * per[3] : nullptr,
        dev[4] ? reinterpret_cast<int*>(dev[4]) + off : nullptr);
    TFS_CUDA(ctx, cudaGetLastError());
    ctx->launches += 1;
  }
  if (any_host) {
    for (int i = 0; i < 5; ++i)
      if (host_out[i])
        TFS_CUDA(ctx, cudaMemcpyAsync(user[i], dev[i], (size_t)n * per[i] * sizeof(float), cudaMemcpyDeviceToHost, st));
    unsigned long long bad = 0;
    TFS_CUDA(ctx, cudaMemcpyAsync(&bad, ctx->bad, sizeof(bad), cudaMemcpyDeviceToHost, st));
    TFS_CUDA(ctx, cudaStreamSynchronize(st));
    ctx->bad_host = (long long)bad;
  } else {
    ctx->bad_host = -1;     // not known yet: tfs_bad_param_count synchronises and reads it on demand
    if (!is_device_ptr(params) || (transfer && !is_device_ptr(transfer)))
      TFS_CUDA(ctx, cudaStreamSynchronize(st));            // host input buffers may be reused
  }
  return TFS_OK;
}

}  // namespace

extern "C" {

int tfs_eval(tfs_ctx* ctx, const double* params, long long n, int N_seg, float* upsilon, float* seg_power,
             float* seg_dh, float* seg_hh, void* stream) {
  return eval_impl(ctx, params, n, N_seg, nullptr, 0, 0.0, 0.0, upsilon, seg_power, seg_dh, seg_hh, stream, "tfs_eval");
}

int tfs_eval_tf(tfs_ctx* ctx, const double* params, long long n, int N_seg, const float* transfer, int n_knots,
                double f_knot0, double f_knot_step, float* upsilon, float* seg_power, float* seg_dh, float* seg_hh,
                void* stream) {
  if (ctx && !transfer) return fail(ctx, TFS_EINVAL, "tfs_eval_tf: transfer is NULL (use tfs_eval for constant factors)");
  return eval_impl(ctx, params, n, N_seg, transfer, n_knots, f_knot0, f_knot_step, upsilon, seg_power, seg_dh, seg_hh, stream,
                   "tfs_eval_tf");
}

int tfs_eval_tseg(tfs_ctx* ctx, const double* params, long long n, int seg_tranches, float* upsilon, int* n_seg_eff,
                  float* seg_power, float* seg_dh, float* seg_hh, void* stream) {
  if (ctx && seg_tranches < 1) return fail(ctx, TFS_EINVAL, "tfs_eval_tseg: seg_tranches must be >= 1 (got %d)", seg_tranches);
  return eval_impl(ctx, params, n, 1, nullptr, 0, 0.0, 0.0, upsilon, seg_power, seg_dh, seg_hh, stream, "tfs_eval_tseg",
                   seg_tranches, n_seg_eff);
}

int tfs_count_pixels(tfs_ctx* ctx, const double* params, long long n, long long* counts, void* stream) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_count_pixels: ctx is NULL");
  if (n < 0) return fail(ctx, TFS_EINVAL, "tfs_count_pixels: n < 0");
  if (!ctx->uploaded) return fail(ctx, TFS_ESTATE, "tfs_count_pixels: no data uploaded (the gap mask is part of the data)");
  if (int rcd = check_device(ctx, "tfs_count_pixels")) return rcd;
  if (n == 0) return TFS_OK;
  if (!params || !counts) return fail(ctx, TFS_EINVAL, "tfs_count_pixels: params and counts are required");
  cudaStream_t st = (cudaStream_t)stream;
  const double* d_params = nullptr;
  int rc = stage_params(ctx, params, n, st, &d_params);
  if (rc) return rc;
  long long* d_counts = counts;
  const bool host = !is_device_ptr(counts);
  if (host) {
    rc = ensure(ctx, &ctx->buf_counts, &ctx->cap_counts, (size_t)n * sizeof(long long));
    if (rc) return rc;
    d_counts = (long long*)ctx->buf_counts;
  }
  EvalArgs a = base_args(ctx);
  a.params = d_params;
  a.n = n;
  const int threads = 256;
  const long long blocks = (n * 32 + threads - 1) / threads;
  if (ctx->opts.basis == 1) count_pixels_wdm_kernel<<<(unsigned)blocks, threads, 0, st>>>(a, d_counts);
  else count_pixels_kernel<<<(unsigned)blocks, threads, 0, st>>>(a, d_counts);
  TFS_CUDA(ctx, cudaGetLastError());
  ctx->launches += 1;
  if (host) {
    TFS_CUDA(ctx, cudaMemcpyAsync(counts, d_counts, (size_t)n * sizeof(long long), cudaMemcpyDeviceToHost, st));
    TFS_CUDA(ctx, cudaStreamSynchronize(st));
  } else if (!is_device_ptr(params)) {
    TFS_CUDA(ctx, cudaStreamSynchronize(st));
  }
  return TFS_OK;
}

int tfs_refine(tfs_ctx* ctx, const double* params, long long n, const long long* idx, long long k, int r,
               double d_mc_rel, double d_tc, double* children, void* stream) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_refine: ctx is NULL");
  if (n < 0 || k < 0) return fail(ctx, TFS_EINVAL, "tfs_refine: n < 0 or k < 0");
  if (r < 1 || r > 64) return fail(ctx, TFS_EINVAL, "tfs_refine: need 1 <= r <= 64 (got %d)", r);
  if (!std::isfinite(d_mc_rel) || !std::isfinite(d_tc)) return fail(ctx, TFS_EINVAL, "tfs_refine: steps must be finite");
  if (int rcd = check_device(ctx, "tfs_refine")) return rcd;
  if (k == 0) return TFS_OK;
  if (!params || !idx || !children) return fail(ctx, TFS_EINVAL, "tfs_refine: params, idx and children are required");
  if (k * (long long)r * r >= (1ll << 32)) return fail(ctx, TFS_EINVAL, "tfs_refine: k*r*r must be < 2^32");
  cudaStream_t st = (cudaStream_t)stream;
  const long long nc = k * (long long)r * r;
  const double* d_params = nullptr;
  int rc = stage_params(ctx, params, n, st, &d_params);
  if (rc) return rc;
  const long long* d_idx = idx;
  const bool host_idx = !is_device_ptr(idx), host_out = !is_device_ptr(children);
  if (host_idx) {
    rc = ensure(ctx, &ctx->buf_tk_idx, &ctx->cap_tk_idx, (size_t)k * sizeof(long long));
    if (rc) return rc;
    TFS_CUDA(ctx, cudaMemcpyAsync(ctx->buf_tk_idx, idx, (size_t)k * sizeof(long long), cudaMemcpyHostToDevice, st));
    d_idx = (const long long*)ctx->buf_tk_idx;
  }
  double* d_out = children;
  if (host_out) {
    rc = ensure(ctx, &ctx->buf_children, &ctx->cap_children, (size_t)nc * TFS_PARAM_COLS * sizeof(double));
    if (rc) return rc;
    d_out = (double*)ctx->buf_children;
  }
  const int threads = 256;
  refine_kernel<<<(unsigned)((nc + threads - 1) / threads), threads, 0, st>>>(d_params, n, d_idx, k, r, d_mc_rel, d_tc, d_out);
  TFS_CUDA(ctx, cudaGetLastError());
  ctx->launches += 1;
  if (host_out)
    TFS_CUDA(ctx, cudaMemcpyAsync(children, d_out, (size_t)nc * TFS_PARAM_COLS * sizeof(double), cudaMemcpyDeviceToHost, st));
  if (host_out || host_idx || !is_device_ptr(params)) TFS_CUDA(ctx, cudaStreamSynchronize(st));
  return TFS_OK;
}

int tfs_tile_lattice(tfs_ctx* ctx, double mc_lo, double mc_hi, int n_mc, double fin_lo, double fin_hi, int n_fin,
                     const double* row, double* params, void* stream) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_tile_lattice: ctx is NULL");
  if (n_mc < 1 || n_fin < 1 || (long long)n_mc * n_fin >= (1ll << 31))
    return fail(ctx, TFS_EINVAL, "tfs_tile_lattice: need n_mc, n_fin >= 1 and n_mc*n_fin < 2^31");
  if (!(mc_lo > 0.0) || !(mc_hi >= mc_lo) || !(fin_lo > 0.0) || !(fin_hi >= fin_lo) || !std::isfinite(mc_hi) || !std::isfinite(fin_hi))
    return fail(ctx, TFS_EINVAL, "tfs_tile_lattice: need 0 < mc_lo <= mc_hi and 0 < fin_lo <= fin_hi (finite)");
  if (!row || !params) return fail(ctx, TFS_EINVAL, "tfs_tile_lattice: row and params are required");
  if (is_device_ptr(row)) return fail(ctx, TFS_EINVAL, "tfs_tile_lattice: row must be a host pointer (8 doubles)");
  if (int rcd = check_device(ctx, "tfs_tile_lattice")) return rcd;
  cudaStream_t st = (cudaStream_t)stream;
  const long long nc = (long long)n_mc * n_fin;
  Row8 r8;
  for (int c = 0; c < 8; ++c) r8.v[c] = row[c];
  const double d_mc = (mc_hi - mc_lo) / (double)n_mc, d_fin = (fin_hi - fin_lo) / (double)n_fin;
  const bool host_out = !is_device_ptr(params);
  double* d_out = params;
  if (host_out) {
    int rc = ensure(ctx, &ctx->buf_children, &ctx->cap_children, (size_t)nc * TFS_PARAM_COLS * sizeof(double));
    if (rc) return rc;
    d_out = (double*)ctx->buf_children;
  }
  tile_lattice_kernel<<<(unsigned)((nc + 255) / 256), 256, 0, st>>>(mc_lo, d_mc, n_mc, fin_lo, d_fin, n_fin, r8, d_out);
  TFS_CUDA(ctx, cudaGetLastError());
  ctx->launches += 1;
  if (host_out) {
    TFS_CUDA(ctx, cudaMemcpyAsync(params, d_out, (size_t)nc * TFS_PARAM_COLS * sizeof(double), cudaMemcpyDeviceToHost, st));
    TFS_CUDA(ctx, cudaStreamSynchronize(st));
  }
  return TFS_OK;
}

int tfs_refine_fin(tfs_ctx* ctx, const double* params, long long n, const long long* idx, long long k, int r,
                   double d_mc, double d_fin, double* children, void* stream) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_refine_fin: ctx is NULL");
  if (n < 0 || k < 0) return fail(ctx, TFS_EINVAL, "tfs_refine_fin: n < 0 or k < 0");
  if (r < 1 || r > 64) return fail(ctx, TFS_EINVAL, "tfs_refine_fin: need 1 <= r <= 64 (got %d)", r);
  if (!std::isfinite(d_mc) || !std::isfinite(d_fin)) return fail(ctx, TFS_EINVAL, "tfs_refine_fin: steps must be finite");
  if (int rcd = check_device(ctx, "tfs_refine_fin")) return rcd;
  if (k == 0) return TFS_OK;
  if (!params || !idx || !children) return fail(ctx, TFS_EINVAL, "tfs_refine_fin: params, idx and children are required");
  if (k * (long long)r * r >= (1ll << 32)) return fail(ctx, TFS_EINVAL, "tfs_refine_fin: k*r*r must be < 2^32");
  cudaStream_t st = (cudaStream_t)stream;
  const long long nc = k * (long long)r * r;
  const double* d_params = nullptr;
  int rc = stage_params(ctx, params, n, st, &d_params);
  if (rc) return rc;
  const long long* d_idx = idx;
  const bool host_idx = !is_device_ptr(idx), host_out = !is_device_ptr(children);
  if (host_idx) {
    rc = ensure(ctx, &ctx->buf_tk_idx, &ctx->cap_tk_idx, (size_t)k * sizeof(long long));
    if (rc) return rc;
    TFS_CUDA(ctx, cudaMemcpyAsync(ctx->buf_tk_idx, idx, (size_t)k * sizeof(long long), cudaMemcpyHostToDevice, st));
    d_idx = (const long long*)ctx->buf_tk_idx;
  }
  double* d_out = children;
  if (host_out) {
    rc = ensure(ctx, &ctx->buf_children, &ctx->cap_children, (size_t)nc * TFS_PARAM_COLS * sizeof(double));
    if (rc) return rc;
    d_out = (double*)ctx->buf_children;
  }
  refine_fin_kernel<<<(unsigned)((nc + 255) / 256), 256, 0, st>>>(d_params, n, d_idx, k, r, d_mc, d_fin, d_out);
  TFS_CUDA(ctx, cudaGetLastError());
  ctx->launches += 1;
  if (host_out)
    TFS_CUDA(ctx, cudaMemcpyAsync(children, d_out, (size_t)nc * TFS_PARAM_COLS * sizeof(double), cudaMemcpyDeviceToHost, st));
  if (host_out || host_idx || !is_device_ptr(params)) TFS_CUDA(ctx, cudaStreamSynchronize(st));
  return TFS_OK;
}

int tfs_probe_l2_bandwidth(tfs_ctx* ctx, long long bytes, int iters, double* gb_per_s, void* stream) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_probe_l2_bandwidth: ctx is NULL");
  if (bytes < (1 << 20) || bytes > (1ll << 32) || iters < 1 || iters > 100000 || !gb_per_s)
    return fail(ctx, TFS_EINVAL, "tfs_probe_l2_bandwidth: need 1 MiB <= bytes <= 4 GiB, 1 <= iters <= 1e5, gb_per_s != NULL");
  cudaStream_t st = (cudaStream_t)stream;
  void* buf = nullptr;
  float* sink = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  const long long n_vec = bytes / 16;
  int rc = TFS_OK;
  cudaError_t e;
  auto done = [&](int code, const char* what, cudaError_t err) {
    if (code) fail(ctx, code, "tfs_probe_l2_bandwidth: %s: %s", what, cudaGetErrorString(err));
    if (buf) cudaFree(buf);
    if (sink) cudaFree(sink);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    return code;
  };
  if ((e = cudaMalloc(&buf, (size_t)n_vec * 16)) != cudaSuccess) return done(TFS_ENOMEM, "cudaMalloc", e);
  if ((e = cudaMalloc((void**)&sink, sizeof(float))) != cudaSuccess) return done(TFS_ENOMEM, "cudaMalloc", e);
  if ((e = cudaMemsetAsync(buf, 0, (size_t)n_vec * 16, st)) != cudaSuccess) return done(TFS_ECUDA, "cudaMemsetAsync", e);
  if ((e = cudaEventCreate(&e0)) != cudaSuccess || (e = cudaEventCreate(&e1)) != cudaSuccess)
    return done(TFS_ECUDA, "cudaEventCreate", e);
  l2_probe_kernel<<<ctx->sm_count, 1024, 0, st>>>((const float4*)buf, n_vec, 2, sink);        // warm the L2
  cudaEventRecord(e0, st);
  l2_probe_kernel<<<ctx->sm_count, 1024, 0, st>>>((const float4*)buf, n_vec, iters, sink);
  cudaEventRecord(e1, st);
  ctx->launches += 2;
  if ((e = cudaEventSynchronize(e1)) != cudaSuccess) return done(TFS_ECUDA, "l2_probe_kernel", e);
  float ms = 0.f;
  if ((e = cudaEventElapsedTime(&ms, e0, e1)) != cudaSuccess) return done(TFS_ECUDA, "cudaEventElapsedTime", e);
  *gb_per_s = (double)n_vec * 16.0 * iters / (ms * 1e-3) / 1e9;
  return done(rc, "", cudaSuccess);
}

int tfs_set_third_channel_factor(tfs_ctx* ctx, double re, double im) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_set_third_channel_factor: ctx is NULL");
  if (ctx->C != 3) return fail(ctx, TFS_EINVAL, "tfs_set_third_channel_factor: the context has %d channels, not 3", ctx->C);
  if (!std::isfinite(re) || !std::isfinite(im)) return fail(ctx, TFS_EINVAL, "tfs_set_third_channel_factor: the factor must be finite");
  ctx->t3[0] = re; ctx->t3[1] = im; ctx->t3_set = true;
  return TFS_OK;
}

int tfs_probe_fp32_issue(tfs_ctx* ctx, int iters, double* scalar_ipc, double* packed_ipc, void* stream) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_probe_fp32_issue: ctx is NULL");
  if (iters < 1 || iters > (1 << 24)) return fail(ctx, TFS_EINVAL, "tfs_probe_fp32_issue: need 1 <= iters <= 2^24");
  int rc = check_device(ctx, "tfs_probe_fp32_issue");
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int nb = ctx->sm_count;
  unsigned long long* d_cyc = nullptr;
  float* d_sink = nullptr;
  cudaError_t e;
  auto done = [&](int code, const char* what, cudaError_t err) {
    if (d_cyc) cudaFree(d_cyc);
    if (d_sink) cudaFree(d_sink);
    return code == TFS_OK ? TFS_OK : fail(ctx, code, "tfs_probe_fp32_issue: %s failed: %s", what, cudaGetErrorString(err));
  };
  if ((e = cudaMalloc((void**)&d_cyc, (size_t)nb * sizeof(unsigned long long))) != cudaSuccess) return done(TFS_ENOMEM, "cudaMalloc", e);
  if ((e = cudaMalloc((void**)&d_sink, sizeof(float))) != cudaSuccess) return done(TFS_ENOMEM, "cudaMalloc", e);
  std::vector<unsigned long long> h((size_t)nb);
  double out[2] = {0.0, 0.0};
  for (int packed = 0; packed < 2; ++packed) {
    fp32_issue_probe_kernel<<<nb, 1024, 0, st>>>(iters / 8 + 1, packed, d_sink, d_cyc);      // warm-up
    fp32_issue_probe_kernel<<<nb, 1024, 0, st>>>(iters, packed, d_sink, d_cyc);
    ctx->launches += 2;
    if ((e = cudaGetLastError()) != cudaSuccess) return done(TFS_ECUDA, "fp32_issue_probe_kernel", e);
    if ((e = cudaMemcpyAsync(h.data(), d_cyc, (size_t)nb * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess)
      return done(TFS_ECUDA, "fp32_issue_probe_kernel", e);
    std::sort(h.begin(), h.end());
    const double cyc = (double)h[h.size() / 2];                       // median SM
    out[packed] = 32.0 * kProbeChains * (double)iters / cyc;           // warp instructions per clock per SM
  }
  if (scalar_ipc) *scalar_ipc = out[0];
  if (packed_ipc) *packed_ipc = out[1];
  return done(TFS_OK, "", cudaSuccess);
}

int tfs_topk(tfs_ctx* ctx, const float* upsilon, long long n, int k, long long* idx, float* val, void* stream) {
  if (!ctx) return fail(nullptr, TFS_EINVAL, "tfs_topk: ctx is NULL");
  if (!upsilon || !idx || !val) return fail(ctx, TFS_EINVAL, "tfs_topk: upsilon, idx and val are required");
  if (n < 1 || n >= (1ll << 32)) return fail(ctx, TFS_EINVAL, "tfs_topk: need 1 <= n < 2^32");
  if (k < 1 || k > n) return fail(ctx, TFS_EINVAL, "tfs_topk: need 1 <= k <= n (got k %d, n %lld)", k, n);
  cudaStream_t st = (cudaStream_t)stream;
  int rc = check_device(ctx, "tfs_topk");
  if (rc) return rc;
  const float* d_in = upsilon;
  if (!is_device_ptr(upsilon)) {
    rc = ensure(ctx, &ctx->buf_tk_in, &ctx->cap_tk_in, (size_t)n * sizeof(float));
    if (rc) return rc;
    TFS_CUDA(ctx, cudaMemcpyAsync(ctx->buf_tk_in, upsilon, (size_t)n * sizeof(float), cudaMemcpyHostToDevice, st));
    d_in = (const float*)ctx->buf_tk_in;
  }
  unsigned P = 1;
  while (P < (unsigned)k) P <<= 1;
  rc = ensure(ctx, &ctx->buf_keys, &ctx->cap_keys, (size_t)P * sizeof(unsigned long long));
  if (rc) return rc;
  unsigned long long* keys = (unsigned long long*)ctx->buf_keys;
  long long* d_idx = idx;
  float* d_val = val;
  const bool host_idx = !is_device_ptr(idx), host_val = !is_device_ptr(val);
  if (host_idx) {
    rc = ensure(ctx, &ctx->buf_tk_idx, &ctx->cap_tk_idx, (size_t)k * sizeof(long long));
    if (rc) return rc;
    d_idx = (long long*)ctx->buf_tk_idx;
  }
  if (host_val) {
    rc = ensure(ctx, &ctx->buf_tk_val, &ctx->cap_tk_val, (size_t)k * sizeof(float));
    if (rc) return rc;
    d_val = (float*)ctx->buf_tk_val;
  }
  const int threads = 256;
  if (n <= (long long)kBitonicBlock) {
    // small batch: select, sort and emit in one launch (the radix select below is 20+ launches: launch-bound here)
    topk_small_kernel<<<1, 1024, 0, st>>>(d_in, (int)n, k, d_idx, d_val);
    ctx->launches += 1;
    TFS_CUDA(ctx, cudaGetLastError());
    if (host_idx) TFS_CUDA(ctx, cudaMemcpyAsync(idx, d_idx, (size_t)k * sizeof(long long), cudaMemcpyDeviceToHost, st));
    if (host_val) TFS_CUDA(ctx, cudaMemcpyAsync(val, d_val, (size_t)k * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (host_idx || host_val || !is_device_ptr(upsilon)) TFS_CUDA(ctx, cudaStreamSynchronize(st));
    return TFS_OK;
  }
  const unsigned blocks = (unsigned)std::min<long long>((n + threads - 1) / threads, (long long)ctx->sm_count * 8);
  topk_init_kernel<<<1, 256, 0, st>>>(ctx->sel, (unsigned long long)k);
  ctx->launches += 1 + 16 + 1 + 1;   // init, 8 x (hist, pick), gather, emit
  for (int pass = 0; pass < 8; ++pass) {
    topk_hist_kernel<<<blocks, threads, 0, st>>>(d_in, n, pass, ctx->sel);
    topk_pick_kernel<<<1, 256, 0, st>>>(pass, ctx->sel);
  }
  topk_gather_kernel<<<blocks, threads, 0, st>>>(d_in, n, ctx->sel, keys, (unsigned)k);
  if (P > (unsigned)k) {
    topk_pad_kernel<<<(P - k + threads - 1) / threads, threads, 0, st>>>(keys, (unsigned)k, P);
    ctx->launches += 1;
  }
  if (P <= 4096) {
    bitonic_small_kernel<<<1, 1024, P * sizeof(unsigned long long), st>>>(keys, P);
    ctx->launches += 1;
  } else {
    // sizes up to the block: one launch; larger sizes: the strides that leave a block one by one, the rest per block
    bitonic_block_kernel<<<P / kBitonicBlock, 1024, 0, st>>>(keys, 2u, kBitonicBlock);
    ctx->launches += 1;
    for (unsigned size = 2 * kBitonicBlock; size <= P && size != 0; size <<= 1) {
      for (unsigned stride = size >> 1; stride > kBitonicBlock / 2; stride >>= 1) {
        bitonic_step_kernel<<<(P / 2 + threads - 1) / threads, threads, 0, st>>>(keys, P, size, stride);
        ctx->launches += 1;
      }
      bitonic_block_kernel<<<P / kBitonicBlock, 1024, 0, st>>>(keys, size, size);
      ctx->launches += 1;
    }
  }
  topk_emit_kernel<<<(k + threads - 1) / threads, threads, 0, st>>>(keys, d_in, k, d_idx, d_val);
  TFS_CUDA(ctx, cudaGetLastError());
  if (host_idx) TFS_CUDA(ctx, cudaMemcpyAsync(idx, d_idx, (size_t)k * sizeof(long long), cudaMemcpyDeviceToHost, st));
  if (host_val) TFS_CUDA(ctx, cudaMemcpyAsync(val, d_val, (size_t)k * sizeof(float), cudaMemcpyDeviceToHost, st));
  if (host_idx || host_val || !is_device_ptr(upsilon)) TFS_CUDA(ctx, cudaStreamSynchronize(st));
  return TFS_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// tfs_topk_static: tfs_topk without a context and without any device allocation (include/tfs.h).
//
// Some users of this library run where they may not allocate on the device: a plug-in inside a host application
// that hands out a fixed memory budget, a real-time loop that cannot afford cudaMalloc's device-wide
// synchronisation, a process whose pool is exhausted.  For them the select's scratch (radix state + sort keys) is
// the fixed array below, part of the library image on every GPU that loads it.
//
// `g_topk_static_scratch` is a DEVICE symbol.  In host code its name is only a host-side shadow of the symbol:
// handing `g_topk_static_scratch` (or &g_topk_static_scratch[0]) to a kernel would pass a host address, which
// faults or -- on systems where the GPU can reach host memory -- quietly scribbles over the wrong bytes.  The
// usable device address comes from cudaGetSymbolAddress, asked once per device with that device current.
// ---------------------------------------------------------------------------------------------
namespace {

constexpr size_t kStaticStateBytes = 2048;   // SelectState (1048 B) rounded up so that the keys stay 256-byte aligned
constexpr size_t kStaticScratchBytes = kStaticStateBytes + (size_t)TFS_TOPK_STATIC_MAX_K * sizeof(unsigned long long);
static_assert(sizeof(SelectState) <= kStaticStateBytes, "SelectState outgrew its slot in the static scratch");
static_assert((TFS_TOPK_STATIC_MAX_K & (TFS_TOPK_STATIC_MAX_K - 1)) == 0, "the key area must hold a power of two");

}  // namespace

static __device__ __align__(256) unsigned char g_topk_static_scratch[kStaticScratchBytes];

namespace {

constexpr int kStaticMaxDevices = 64;
struct StaticSlot { unsigned char* base = nullptr; int sm_count = 0; };
StaticSlot g_static_slot[kStaticMaxDevices];
std::mutex g_static_mutex;

// Device address of the scratch on the CURRENT device (looked up on the first call per device, cached afterwards).
int static_scratch(int* device_out, StaticSlot* out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cudaGetLastError(); return fail(nullptr, TFS_ECUDA, "tfs_topk_static: cudaGetDevice failed: %s", cudaGetErrorString(e)); }
  if (dev < 0 || dev >= kStaticMaxDevices) return fail(nullptr, TFS_EINVAL, "tfs_topk_static: device ordinal %d not supported (< %d)", dev, kStaticMaxDevices);
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticSlot& s = g_static_slot[dev];
  if (!s.base) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_topk_static_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return fail(nullptr, TFS_ECUDA, "tfs_topk_static: cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
    }
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess || sms < 1) {
      cudaGetLastError();
      return fail(nullptr, TFS_ECUDA, "tfs_topk_static: cudaDeviceGetAttribute failed on device %d: %s", dev, cudaGetErrorString(e));
    }
    s.sm_count = sms;
    s.base = (unsigned char*)p;
  }
  *device_out = dev;
  *out = s;
  return TFS_OK;
}

// device memory that belongs to `dev` (managed memory is accepted as well)
bool is_device_ptr_on(const void* p, int dev) {
  cudaPointerAttributes at;
  cudaError_t e = cudaPointerGetAttributes(&at, p);
  if (e != cudaSuccess) { cudaGetLastError(); return false; }
  if (at.type == cudaMemoryTypeManaged) return true;
  return at.type == cudaMemoryTypeDevice && at.device == dev;
}

}  // namespace

extern "C" int tfs_topk_static(const float* upsilon, long long n, int k, long long* idx, float* val, void* stream) {
  if (!upsilon || !idx || !val) return fail(nullptr, TFS_EINVAL, "tfs_topk_static: upsilon, idx and val are required");
  if (n < 1 || n >= (1ll << 32)) return fail(nullptr, TFS_EINVAL, "tfs_topk_static: need 1 <= n < 2^32");
  if (k < 1 || k > n) return fail(nullptr, TFS_EINVAL, "tfs_topk_static: need 1 <= k <= n (got k %d, n %lld)", k, n);
  if (k > TFS_TOPK_STATIC_MAX_K)
    return fail(nullptr, TFS_EINVAL, "tfs_topk_static: k = %d exceeds TFS_TOPK_STATIC_MAX_K = %d, the size of the built-in "
                                     "scratch (use tfs_topk, which allocates)", k, TFS_TOPK_STATIC_MAX_K);
  int dev = -1;
  StaticSlot slot;
  int rc = static_scratch(&dev, &slot);
  if (rc) return rc;
  if (!is_device_ptr_on(upsilon, dev) || !is_device_ptr_on(idx, dev) || !is_device_ptr_on(val, dev))
    return fail(nullptr, TFS_EINVAL, "tfs_topk_static: upsilon, idx and val must be device pointers on the current device "
                                     "(staging a host buffer would need an allocation)");
  cudaStream_t st = (cudaStream_t)stream;
  SelectState* sel = (SelectState*)slot.base;
  unsigned long long* keys = (unsigned long long*)(slot.base + kStaticStateBytes);
  auto launched = [&](const char* what) {
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? TFS_OK : fail(nullptr, TFS_ECUDA, "tfs_topk_static: %s failed: %s", what, cudaGetErrorString(e));
  };
  const int threads = 256;
  if (n <= (long long)kBitonicBlock) {       // whole select in shared memory, as in tfs_topk: the scratch is not touched
    topk_small_kernel<<<1, 1024, 0, st>>>(upsilon, (int)n, k, idx, val);
    return launched("topk_small_kernel");
  }
  unsigned P = 1;
  while (P < (unsigned)k) P <<= 1;           // <= TFS_TOPK_STATIC_MAX_K: fits the key area
  const unsigned blocks = (unsigned)std::min<long long>((n + threads - 1) / threads, (long long)slot.sm_count * 8);
  topk_init_kernel<<<1, 256, 0, st>>>(sel, (unsigned long long)k);      // zeroes prefix, rank, counter and histogram left by the last call
  for (int pass = 0; pass < 8; ++pass) {
    topk_hist_kernel<<<blocks, threads, 0, st>>>(upsilon, n, pass, sel);
    topk_pick_kernel<<<1, 256, 0, st>>>(pass, sel);
  }
  topk_gather_kernel<<<blocks, threads, 0, st>>>(upsilon, n, sel, keys, (unsigned)k);     // writes keys[0, k)
  if (P > (unsigned)k) topk_pad_kernel<<<(P - k + threads - 1) / threads, threads, 0, st>>>(keys, (unsigned)k, P);   // and [k, P)
  if (P <= 4096) {
    bitonic_small_kernel<<<1, 1024, P * sizeof(unsigned long long), st>>>(keys, P);
  } else {
    bitonic_block_kernel<<<P / kBitonicBlock, 1024, 0, st>>>(keys, 2u, kBitonicBlock);
    for (unsigned size = 2 * kBitonicBlock; size <= P && size != 0; size <<= 1) {
      for (unsigned stride = size >> 1; stride > kBitonicBlock / 2; stride >>= 1)
        bitonic_step_kernel<<<(P / 2 + threads - 1) / threads, threads, 0, st>>>(keys, P, size, stride);
      bitonic_block_kernel<<<P / kBitonicBlock, 1024, 0, st>>>(keys, size, size);
    }
  }
  topk_emit_kernel<<<(k + threads - 1) / threads, threads, 0, st>>>(keys, upsilon, k, idx, val);
  return launched("top-k kernels");
}
