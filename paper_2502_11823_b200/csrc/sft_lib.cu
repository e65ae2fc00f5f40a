// sft_lib.cu - host side of libsft_b200.so: the C ABI of include/sft.h.  Argument checking,
// device-memory ownership, launch geometry; all arithmetic of the method is in sft_kernels.cuh.
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <vector>
#include <mutex>
#include <utility>

#include "../../include/sft.h"
#include "sft_kernels.cuh"
#include "sft_launch.cuh"
#include "alu_peaks.cuh"
#include "sft_ingest.cuh"

#define SFT_API extern "C" __attribute__((visibility("default")))

using sftk::KParams;

struct sft_plan {
  sft_plan_desc d;
  int nb = 0;             // stored bins per SFT
  int n_samp = 0;         // samples per SFT
  int kv_lo = 0, kv_hi = 0;
  cudaStream_t stream = nullptr;
  int PAD = 0, npair = 0; // zero padding (bins) on both sides of a stored row; 16-byte pair entries per row
  float4 *Dp = nullptr;   // [2][C][n_sft][npair] pair-planar whitened data, two parities (sft_kernels.cuh)
  float2 *ubp = nullptr;  // [2][C][npair]
  float *us2 = nullptr;   // [C][n_sft]
  float2 *rtab = nullptr; // [C][n_sft]
  double sigma[SFT_MAX_CHANNELS] = {0, 0, 0, 0};
  double s_ref[SFT_MAX_CHANNELS] = {1, 1, 1, 1};       // reference PSD level of the channel's shape (sft_load_data)
  double *shape_dev = nullptr;                         // [C][nb] device copy of the PSD shapes (sft_append_sfts reuses them)
  bool has_shape[SFT_MAX_CHANNELS] = {false, false, false, false};
  bool loaded[SFT_MAX_CHANNELS] = {false, false, false, false};
  // scratch, grown on demand
  double *part = nullptr; size_t part_bytes = 0;
  double *d_params = nullptr; size_t params_bytes = 0;
  void *d_out = nullptr; size_t out_bytes = 0;         // staging for host outputs
  void *h_pin = nullptr; size_t pin_bytes = 0;         // pinned host staging (params in, result vectors out)
  void *scan = nullptr; size_t scan_bytes = 0;         // cumulative: look-back records {aggregate, inclusive} per (unit, template), 16 bytes each
  unsigned epoch = 0;                                  // 16-bit tag of the entries published by the current cumulative call (1 ... 65534)
  double *td = nullptr; size_t td_bytes = 0;           // per-template constants (sft_tmpl_kernel)
  float *tf = nullptr; size_t tf_bytes = 0;
  float4 *mtab = nullptr;                              // [C][n_sft][n_node][4] data-moment table (sft_table.cuh), or null
  float4 *htab = nullptr;                              // [C][n_kc * HTAB_R][4] <h,h> table
  float4 *htab1 = nullptr;                             // [C][n_kc * HT1_R] compact tier-1 <h,h> table
  float2 *ptab = nullptr;                              // [(2K+1)][TAB_R][TAB_Q+1] kernel moments at the nodes
  int n_kc = 0, n_node = 0;
  int4 *tblk = nullptr;                                // [ceil(n_sft/32)] layout of the moment table per block of 32 SFT slots (sft_kernels.cuh)
  size_t m_f4_chan = 0;                                // float4 entries of mtab per channel
  int w_max = 0;                                       // widest block (window positions)
  bool banded = false;                                 // layout from sft_plan_set_table_track
  int *counter = nullptr;                              // work-unit counter of the persistent main kernel
  unsigned *chk = nullptr;                             // checked build only (SFT_CHECKED): first failing bounds-check site
  unsigned long long *path_counts = nullptr;           // [PATH_N] diagnostic counters
  int n_sm = 0;
  int chunk_user = 0;
  long long slab_user = 0;                             // sft_plan_set_host_slab: templates per slab of the host-output pipeline (0 = auto)
  cudaStream_t copy_stream = nullptr;                  // sft_cumulative_snr with host outputs: device-to-host copies of finished slabs
  cudaEvent_t ev_slab[2] = {nullptr, nullptr};
  long long launches = 0;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  bool timed = false;
  char err[512] = {0};
};

static thread_local char g_create_err[512] = {0};

static sft_status fail(sft_plan *p, sft_status st, const char *fmt, ...) {
  char *buf = p ? p->err : g_create_err;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, 512, fmt, ap);
  va_end(ap);
  return st;
}

#define CU(p, call)                                                                         \
  do {                                                                                      \
    cudaError_t e_ = (call);                                                                \
    if (e_ != cudaSuccess)                                                                  \
      return fail(p, e_ == cudaErrorMemoryAllocation ? SFT_ENOMEM : SFT_ECUDA, "%s: %s", #call, \
                  cudaGetErrorString(e_));                                                  \
  } while (0)

static sft_status grow_pinned(sft_plan *p, size_t need) {
  if (p->pin_bytes >= need) return SFT_OK;
  if (p->h_pin) { cudaFreeHost(p->h_pin); p->h_pin = nullptr; p->pin_bytes = 0; }
  cudaError_t e = cudaMallocHost(&p->h_pin, need);
  if (e != cudaSuccess) return fail(p, SFT_ENOMEM, "cudaMallocHost(%zu): %s", need, cudaGetErrorString(e));
  p->pin_bytes = need;
  return SFT_OK;
}

static sft_status grow(sft_plan *p, void **ptr, size_t *have, size_t need) {
  if (*have >= need) return SFT_OK;
  if (*ptr) { CU(p, cudaFree(*ptr)); *ptr = nullptr; *have = 0; }
  CU(p, cudaMalloc(ptr, need));
  *have = need;
  return SFT_OK;
}

#ifdef SFT_CHECKED
SFT_API const char *sft_version(void) { return "sft_b200 0.1 (sm_100a, checked build: bounds tests on)"; }
#else
SFT_API const char *sft_version(void) { return "sft_b200 0.1 (sm_100a)"; }
#endif

SFT_API const char *sft_last_error(const sft_plan *plan) { return plan ? plan->err : g_create_err; }

// Lays out and allocates the data-moment table (replacing any previous one).  `kb` / `w` [n_blocks]: first window position
// (counted from k_lo - K) and number of positions of every block of 32 SFT slots; null = all n_kc positions everywhere.
// SFT_ENOMEM (plan left without a table) if it does not fit in a quarter of the free device memory or in 32-bit indexing.
static sft_status table_layout(sft_plan *p, const int *kb, int /*unused*/, const int *w) {
  const size_t N = p->d.n_sft, C = p->d.n_channels, nblk = (N + 31) / 32, f4_node = (sftk::TAB_Q + 1) / 2;
  std::vector<int4> h(nblk);
  size_t off = 0;
  int wmax = 0;
  for (size_t b = 0; b < nblk; ++b) {
    const int kbb = kb ? kb[b] : 0, wb = w ? w[b] : p->n_kc;
    const size_t rows = (b + 1 < nblk) ? 32 : N - 32 * b, mrow = (size_t)wb * sftk::TAB_R * f4_node;
    if (off + rows * mrow >= 4000000000ull) { off = ~size_t(0) / 2; break; }
    h[b] = make_int4((int)(unsigned)off, kbb, wb, (int)mrow);
    off += rows * mrow;
    if (wb > wmax) wmax = wb;
  }
  cudaFree(p->mtab); p->mtab = nullptr;
  cudaFree(p->tblk); p->tblk = nullptr;
  p->m_f4_chan = 0;
  size_t free_b = 0, total_b = 0;
  cudaMemGetInfo(&free_b, &total_b);
  const double m_bytes = (double)C * (double)off * 16.0;
  if (off >= 4000000000ull || (double)C * (double)off >= 4.0e9 || m_bytes > 0.25 * (double)free_b)
    return fail(p, SFT_ENOMEM, "moment tables of %.3g bytes do not fit (free %.3g)", m_bytes, (double)free_b);
  if (cudaMalloc((void **)&p->mtab, (size_t)m_bytes + 256) != cudaSuccess || cudaMalloc((void **)&p->tblk, nblk * sizeof(int4)) != cudaSuccess) {
    cudaFree(p->mtab); p->mtab = nullptr;
    cudaFree(p->tblk); p->tblk = nullptr;
    cudaGetLastError();
    return fail(p, SFT_ENOMEM, "cudaMalloc of the moment tables (%.3g bytes) failed", m_bytes);
  }
  cudaError_t e = cudaMemcpyAsync(p->tblk, h.data(), nblk * sizeof(int4), cudaMemcpyHostToDevice, p->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);          // (h is a local)
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "table layout copy: %s", cudaGetErrorString(e));
  p->m_f4_chan = off;
  p->w_max = wmax;
  return SFT_OK;
}

SFT_API sft_status sft_plan_create(const sft_plan_desc *desc, sft_plan **out) {
  g_create_err[0] = 0;
  if (!desc || !out) return fail(nullptr, SFT_EINVAL, "sft_plan_create: NULL argument");
  const sft_plan_desc &d = *desc;
  if (d.n_channels < 1 || d.n_channels > SFT_MAX_CHANNELS)
    return fail(nullptr, SFT_EINVAL, "n_channels=%d outside 1..%d", d.n_channels, SFT_MAX_CHANNELS);
  if (d.n_sft < 1 || d.n_sft > (1ll << 30)) return fail(nullptr, SFT_EINVAL, "n_sft=%lld out of range", (long long)d.n_sft);
  if (!(d.t_sft > 0.0) || !(d.fs > 0.0) || !isfinite(d.t0)) return fail(nullptr, SFT_EINVAL, "t_sft, fs must be > 0 and t0 finite");
  const double n = d.t_sft * d.fs;
  if (fabs(n - nearbyint(n)) > 1e-9 * fmax(1.0, n) || n < 2.0 || n > 2e9)
    return fail(nullptr, SFT_ESHAPE, "t_sft*fs = %.12g is not an integer number of samples (P:157)", n);
  if (d.k_lo < 0 || d.k_hi <= d.k_lo) return fail(nullptr, SFT_ESHAPE, "stored band [k_lo=%d, k_hi=%d) is empty or negative", d.k_lo, d.k_hi);
  if (d.K < 0 || d.K > SFT_MAX_K) return fail(nullptr, SFT_EINVAL, "K=%d outside 0..%d", d.K, SFT_MAX_K);
  if (d.kernel != SFT_KERNEL_DIRICHLET && d.kernel != SFT_KERNEL_FRESNEL) return fail(nullptr, SFT_EINVAL, "unknown kernel %d", d.kernel);
  if (d.waveform < SFT_WF_PN0 || d.waveform > SFT_WF_PN15) return fail(nullptr, SFT_EINVAL, "unknown waveform %d", d.waveform);
  if (d.phase_path != SFT_PHASE_FP64 && d.phase_path != SFT_PHASE_SPLIT32) return fail(nullptr, SFT_EINVAL, "unknown phase_path %d", d.phase_path);
  if (d.response < SFT_RESP_NONE || d.response > SFT_RESP_ANNUAL) return fail(nullptr, SFT_EINVAL, "unknown response %d", d.response);
  if (!(d.f_ref > 0.0)) return fail(nullptr, SFT_EINVAL, "f_ref must be > 0");
  if (!(d.f_hi >= d.f_lo)) return fail(nullptr, SFT_EINVAL, "need f_lo <= f_hi");
  if (d.response == SFT_RESP_ANNUAL && !(d.resp_period > 0.0)) return fail(nullptr, SFT_EINVAL, "resp_period must be > 0");
  if (d.include_dc != 0 && d.include_dc != 1) return fail(nullptr, SFT_EINVAL, "include_dc must be 0 or 1");
  if (d.evaluator < SFT_EVAL_AUTO || d.evaluator > SFT_EVAL_TABLE) return fail(nullptr, SFT_EINVAL, "unknown evaluator %d", d.evaluator);
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess) return fail(nullptr, SFT_ECUDA, "cudaGetDeviceCount: %s", cudaGetErrorString(e));
  if (d.device < 0 || d.device >= ndev) return fail(nullptr, SFT_EINVAL, "device %d not in 0..%d", d.device, ndev - 1);
  e = cudaSetDevice(d.device);
  if (e != cudaSuccess) return fail(nullptr, SFT_ECUDA, "cudaSetDevice: %s", cudaGetErrorString(e));

  sft_plan *p = new (std::nothrow) sft_plan();
  if (!p) return fail(nullptr, SFT_ENOMEM, "out of host memory");
  p->d = d;
  p->nb = d.k_hi - d.k_lo;
  p->n_samp = (int)nearbyint(n);
  const int k_first = d.include_dc ? 0 : 1;                             // DESIGN A6: 1 <= k <= n/2-1 (0 <= k with include_dc)
  p->kv_lo = d.k_lo > k_first ? d.k_lo : k_first;
  p->kv_hi = d.k_hi < p->n_samp / 2 ? d.k_hi : p->n_samp / 2;
  p->stream = (cudaStream_t)d.stream;
  const size_t C = d.n_channels, N = d.n_sft, nb = p->nb;
  sft_status st = SFT_OK;
  auto alloc = [&](void **ptr, size_t bytes) {
    if (st != SFT_OK) return;
    cudaError_t e2 = cudaMalloc(ptr, bytes);
    if (e2 != cudaSuccess) st = fail(nullptr, SFT_ENOMEM, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e2));
  };
  p->PAD = 2 * d.K + 2;
  p->npair = (p->nb + 2 * p->PAD + 1) / 2 + 1;
  const size_t npair = p->npair;
  (void)nb;
  if (2.0 * C * (double)N * npair + npair >= 2147483648.0)
    st = fail(nullptr, SFT_EUNSUPPORTED, "data store of %.3g pair entries exceeds 32-bit indexing", 2.0 * C * (double)N * npair);
  alloc((void **)&p->Dp, (2 * C * N + 1) * npair * sizeof(float4));   // + one row: the kernel prefetches one row ahead
  alloc((void **)&p->ubp, 2 * C * npair * sizeof(float2));
  alloc((void **)&p->us2, C * N * sizeof(float));
  alloc((void **)&p->rtab, C * N * sizeof(float2));
  alloc((void **)&p->shape_dev, C * (size_t)p->nb * sizeof(double));
  // moment tables (sft_table.cuh): 64 bytes per node, TAB_R nodes per window position and SFT.  AUTO takes
  // them when they fit in a quarter of the free device memory, TABLE insists, DIRECT never builds them.
  p->n_kc = p->nb + 2 * d.K;
  p->n_node = p->n_kc * sftk::TAB_R;
  if (st == SFT_OK && d.evaluator != SFT_EVAL_DIRECT) {
    st = table_layout(p, nullptr, 0, nullptr);         // every block covers all n_kc window positions
    if (st == SFT_ENOMEM && d.evaluator == SFT_EVAL_AUTO) st = SFT_OK;   // does not fit: direct evaluator (mtab stays null)
    if (st != SFT_OK) memcpy(g_create_err, p->err, 512);
    if (st == SFT_OK) {
      alloc((void **)&p->htab, C * (size_t)p->n_kc * sftk::HTAB_R * sftk::HTAB_W * sizeof(float));
      alloc((void **)&p->htab1, C * (size_t)p->n_kc * sftk::HT1_R * sizeof(float4));
      alloc((void **)&p->ptab, (size_t)(2 * d.K + 1) * sftk::TAB_R * (sftk::TAB_Q + 1) * sizeof(float2));
      if (st == SFT_OK) {
        const int n = (2 * d.K + 1) * sftk::TAB_R;
        sftk::sft_ptab_kernel<<<(n + 63) / 64, 64, 0, p->stream>>>(d.K, p->ptab);
        p->launches++;
        cudaError_t e2 = cudaGetLastError();
        if (e2 != cudaSuccess) st = fail(nullptr, SFT_ECUDA, "kernel-moment table launch: %s", cudaGetErrorString(e2));
      }
    }
  }
  alloc((void **)&p->counter, sizeof(int));
#ifdef SFT_CHECKED
  alloc((void **)&p->chk, sizeof(unsigned));
  if (st == SFT_OK && cudaMemset(p->chk, 0, sizeof(unsigned)) != cudaSuccess) st = fail(nullptr, SFT_ECUDA, "plan set-up: cudaMemset");
#endif
  alloc((void **)&p->path_counts, sftk::PATH_N * sizeof(unsigned long long));
  if (st == SFT_OK) {
    cudaError_t e2 = cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, d.device);
    if (e2 == cudaSuccess) e2 = cudaMemsetAsync(p->path_counts, 0, sftk::PATH_N * sizeof(unsigned long long), p->stream);
    if (e2 != cudaSuccess) st = fail(nullptr, SFT_ECUDA, "plan set-up: %s", cudaGetErrorString(e2));
  }
  if (st == SFT_OK) {
    cudaError_t e2 = cudaEventCreate(&p->ev0);
    if (e2 == cudaSuccess) e2 = cudaEventCreate(&p->ev1);
    if (e2 != cudaSuccess) st = fail(nullptr, SFT_ECUDA, "cudaEventCreate: %s", cudaGetErrorString(e2));
  }
  if (st == SFT_OK && d.response == SFT_RESP_ANNUAL) {
    for (size_t c = 0; c < C; ++c) {
      sftk::sft_annual_table_kernel<<<(unsigned)((N + 255) / 256), 256, 0, p->stream>>>(
          (int)N, d.t0, d.t_sft, d.resp_period, d.resp_psi[c], p->rtab + c * N);
      p->launches++;
    }
    cudaError_t e2 = cudaGetLastError();
    if (e2 != cudaSuccess) st = fail(nullptr, SFT_ECUDA, "annual table launch: %s", cudaGetErrorString(e2));
  }
  if (st != SFT_OK) {
    char keep[512];
    memcpy(keep, g_create_err, 512);
    sft_plan_destroy(p);
    memcpy(g_create_err, keep, 512);
    return st;
  }
  *out = p;
  return SFT_OK;
}

SFT_API sft_status sft_plan_destroy(sft_plan *p) {
  if (!p) return SFT_OK;
  cudaSetDevice(p->d.device);
  cudaStreamSynchronize(p->stream);
  cudaFree(p->Dp); cudaFree(p->ubp); cudaFree(p->us2); cudaFree(p->rtab); cudaFree(p->shape_dev);
  cudaFree(p->part); cudaFree(p->d_params); cudaFree(p->d_out); cudaFree(p->scan);
  if (p->h_pin) cudaFreeHost(p->h_pin);
  cudaFree(p->td); cudaFree(p->tf); cudaFree(p->counter); cudaFree(p->path_counts); cudaFree(p->chk);
  cudaFree(p->mtab); cudaFree(p->htab); cudaFree(p->htab1); cudaFree(p->ptab); cudaFree(p->tblk);
  if (p->copy_stream) { cudaStreamSynchronize(p->copy_stream); cudaStreamDestroy(p->copy_stream); }
  for (int i = 0; i < 2; ++i) if (p->ev_slab[i]) cudaEventDestroy(p->ev_slab[i]);
  if (p->ev0) cudaEventDestroy(p->ev0);
  if (p->ev1) cudaEventDestroy(p->ev1);
  delete p;
  return SFT_OK;
}

SFT_API sft_status sft_plan_sync(sft_plan *p) {
  if (!p) return SFT_EINVAL;
  CU(p, cudaSetDevice(p->d.device));
  CU(p, cudaStreamSynchronize(p->stream));
  return SFT_OK;
}

SFT_API int64_t sft_plan_launch_count(const sft_plan *p) { return p ? p->launches : 0; }

SFT_API double sft_plan_last_kernel_ms(sft_plan *p) {
  if (!p || !p->timed) return -1.0;
  if (cudaSetDevice(p->d.device) != cudaSuccess) return -1.0;
  if (cudaEventSynchronize(p->ev1) != cudaSuccess) return -1.0;
  float ms = -1.f;
  if (cudaEventElapsedTime(&ms, p->ev0, p->ev1) != cudaSuccess) return -1.0;
  return (double)ms;
}

SFT_API sft_status sft_plan_path_counts(sft_plan *p, int64_t *out, int32_t n_out) {
  if (!p) return SFT_EINVAL;
  if (!out || n_out < 1) return fail(p, SFT_EINVAL, "sft_plan_path_counts: out is NULL or n_out < 1");
  CU(p, cudaSetDevice(p->d.device));
  unsigned long long h[sftk::PATH_N];
  CU(p, cudaMemcpyAsync(h, p->path_counts, sizeof(h), cudaMemcpyDeviceToHost, p->stream));
  CU(p, cudaStreamSynchronize(p->stream));
  for (int i = 0; i < n_out && i < sftk::PATH_N; ++i) out[i] = (int64_t)h[i];
  return SFT_OK;
}

// SFT-length rule, Eq.(33)-(34) P:244-248 (host arithmetic only).
SFT_API sft_status sft_tsft_rule(double m_chirp, double eta, int32_t waveform, double f_max, double delta, double *t_sft,
                                 double *fddot_max) {
  g_create_err[0] = 0;
  if (!t_sft) return fail(nullptr, SFT_EINVAL, "sft_tsft_rule: t_sft is NULL");
  if (!(m_chirp > 0.0) || !(eta > 0.0) || !(eta <= 0.25) || !(f_max > 0.0) || !(delta > 0.0))
    return fail(nullptr, SFT_EINVAL, "sft_tsft_rule: need m_chirp, f_max, delta > 0 and 0 < eta <= 1/4");
  if (waveform < SFT_WF_PN0 || waveform > SFT_WF_PN15) return fail(nullptr, SFT_EINVAL, "unknown waveform %d", waveform);
  const double PI = 3.141592653589793;
  const double M = m_chirp * pow(eta, -0.6) * sftk::GMSUN_S;
  const double cf = waveform >= SFT_WF_PN1 ? 743.0 / 2688.0 + 11.0 / 32.0 * eta : 0.0;
  const double c15 = waveform >= SFT_WF_PN15 ? sftk::C15_F : 0.0;
  // Theta at which f(Theta) = Theta^(-3/8) (1 + cf Theta^(-1/4)) / (8 pi M) reaches f_max: f falls monotonically with Theta;
  // start from the 0PN root (where the 1PN f is higher, i.e. the root lies at larger Theta) and use Newton's method in
  // u = Theta^(-1/8):  g(u) = u^3 (1 + cf u^2 + c15 u^3) - 8 pi M f_max
  const double target = 8.0 * PI * M * f_max;
  double u = cbrt(target);
  for (int it = 0; it < 60; ++it) {
    const double u2 = u * u, u3 = u2 * u;
    const double g = u3 * (1.0 + cf * u2 + c15 * u3) - target, dg = 3.0 * u2 + 5.0 * cf * u2 * u2 + 6.0 * c15 * u2 * u3;
    const double un = u - g / dg;
    if (fabs(un - u) <= 1e-15 * fabs(u)) { u = un; break; }
    u = un;
  }
  if (!(u > 0.0) || !isfinite(u)) return fail(nullptr, SFT_EINVAL, "sft_tsft_rule: no root for f_max = %g", f_max);
  // d^2 f / dt^2 = k^2/(8 pi M) [ (3/8)(11/8) Theta^(-19/8) + (5/8)(13/8) cf Theta^(-21/8) ],  k = eta/(5M), Theta^(-1/8) = u
  const double k = eta / (5.0 * M);
  const double u19 = pow(u, 19.0), u21 = u19 * u * u;
  const double fdd = k * k / (8.0 * PI * M) * (0.375 * 1.375 * u19 + 0.625 * 1.625 * cf * u21 + 0.75 * 1.75 * c15 * u21 * u);
  if (fddot_max) *fddot_max = fdd;
  *t_sft = cbrt(2.0 * delta / fdd);
  return SFT_OK;
}

// Moment tables restricted to the band a known track sweeps.  The k_c of the fiducial template at the first and last SFT of
// every block of 32 slots (host double arithmetic of the same closed form as the kernels: DESIGN W1/W2, A5) +- half_width
// bins gives the block's window positions; blocks the fiducial signal does not reach get no rows.
SFT_API sft_status sft_plan_set_table_track(sft_plan *p, const double *fiducial, int32_t half_width) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (p->d.evaluator == SFT_EVAL_DIRECT) return SFT_OK;             // no tables: nothing to lay out
  if (half_width < 0) return fail(p, SFT_EINVAL, "half_width must be >= 0");
  CU(p, cudaSetDevice(p->d.device));
  CU(p, cudaStreamSynchronize(p->stream));
  const size_t N = p->d.n_sft, nblk = (N + 31) / 32;
  std::vector<int> kb, w;
  if (fiducial) {
    kb.assign(nblk, 0);
    w.assign(nblk, 0);
    const double mc = fiducial[0], eta = fiducial[1], tau0 = fiducial[2] - p->d.t0, T = p->d.t_sft;
    if (!(mc > 0.0) || !(eta > 0.0) || !(eta <= 0.25) || !isfinite(tau0)) return fail(p, SFT_EINVAL, "fiducial template: need m_chirp > 0, 0 < eta <= 1/4");
    const double M = mc * pow(eta, -0.6) * sftk::GMSUN_S, k = eta / (5.0 * M), F0T = T / (8.0 * 3.141592653589793 * M);
    const double cf = p->d.waveform >= SFT_WF_PN1 ? 743.0 / 2688.0 + 11.0 / 32.0 * eta : 0.0, c15 = p->d.waveform >= SFT_WF_PN15 ? sftk::C15_F : 0.0;
    auto kc_of = [&](size_t a, long long &kc) {
      const double tau = tau0 - (double)a * T;
      if (!(tau > T)) return false;
      const double q = pow(k * tau, -0.125), q2 = q * q, q3 = q2 * q, q8 = q2 * q2 * q2 * q2;
      const double fT = F0T * q3 * (1.0 + cf * q2 + c15 * q3), b = F0T * k * T * (q8 * q3) * (0.375 + 0.625 * cf * q2 + 0.75 * c15 * q3);
      const double y = p->d.kernel == SFT_KERNEL_FRESNEL ? fT + 0.5 * b : fT;
      if (!isfinite(y) || fabs(y) > 1.0e9) return false;
      kc = (long long)floor(y + 0.5);
      return true;
    };
    const long long base = (long long)p->d.k_lo - p->d.K;                // window position 0
    for (size_t b = 0; b < nblk; ++b) {
      const size_t a0 = 32 * b, a1 = (a0 + 31 < N ? a0 + 31 : N - 1);
      long long k0, k1;
      if (!kc_of(a0, k0)) continue;                                       // ended before the block starts: no rows
      size_t al = a1;
      while (al > a0 && !kc_of(al, k1)) --al;                              // (the signal may end inside the block)
      if (al == a0) k1 = k0;
      long long lo = k0 - half_width - base, hi = k1 + half_width - base;
      if (lo < 0) lo = 0;
      if (hi > p->n_kc - 1) hi = p->n_kc - 1;
      if (hi >= lo) { kb[b] = (int)lo; w[b] = (int)(hi - lo + 1); }
    }
  }
  sft_status st = table_layout(p, fiducial ? kb.data() : nullptr, 0, fiducial ? w.data() : nullptr);
  for (int c = 0; c < p->d.n_channels; ++c) p->loaded[c] = false;        // the tables are gone: sft_load_data again
  p->banded = fiducial != nullptr && st == SFT_OK;
  if (st == SFT_ENOMEM && p->d.evaluator == SFT_EVAL_AUTO) return SFT_OK; // no tables: the direct evaluator serves
  return st;
}

SFT_API int64_t sft_plan_table_bytes(const sft_plan *p) {
  return p && p->mtab ? (int64_t)(p->m_f4_chan * 16 * (size_t)p->d.n_channels) : 0;
}

SFT_API sft_status sft_plan_set_chunk(sft_plan *p, int32_t c) {
  if (!p) return SFT_EINVAL;
  if (c < 0) return fail(p, SFT_EINVAL, "sfts_per_block must be >= 0");
  p->chunk_user = c;
  return SFT_OK;
}

SFT_API sft_status sft_plan_set_host_slab(sft_plan *p, int64_t templates) {
  if (!p) return SFT_EINVAL;
  if (templates < 0) return fail(p, SFT_EINVAL, "templates_per_slab must be >= 0");
  p->slab_user = templates;
  return SFT_OK;
}

SFT_API sft_status sft_load_data(sft_plan *p, int32_t channel, const float *sft_bins, const double *psd_scale,
                                    const double *psd_shape, const float *response, int32_t mem) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (channel < 0 || channel >= p->d.n_channels) return fail(p, SFT_EINVAL, "channel %d outside 0..%d", channel, p->d.n_channels - 1);
  if (!sft_bins || !psd_scale) return fail(p, SFT_EINVAL, "sft_bins and psd_scale are required");
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(p, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  if (p->d.response == SFT_RESP_TABLE && !response) return fail(p, SFT_EINVAL, "response table required by SFT_RESP_TABLE");
  CU(p, cudaSetDevice(p->d.device));
  const size_t N = p->d.n_sft, nb = p->nb;
  // PSD shape on the host: reference level S_ref = min S over the valid stored bins
  std::vector<double> shape;
  double S_ref = 1.0;
  if (psd_shape) {
    shape.resize(nb);
    if (mem == SFT_MEM_DEVICE) {
      CU(p, cudaMemcpyAsync(shape.data(), psd_shape, nb * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
      CU(p, cudaStreamSynchronize(p->stream));
    } else {
      memcpy(shape.data(), psd_shape, nb * sizeof(double));
    }
    S_ref = INFINITY;
    for (size_t j = 0; j < nb; ++j) {
      const int k = p->d.k_lo + (int)j;
      if (k < p->kv_lo || k >= p->kv_hi) continue;
      if (!(shape[j] > 0.0) || !isfinite(shape[j])) return fail(p, SFT_EINVAL, "psd_shape[%zu] = %g is not a positive finite PSD", j, shape[j]);
      if (shape[j] < S_ref) S_ref = shape[j];
    }
    if (!isfinite(S_ref)) S_ref = 1.0;   // no valid bin in the stored band: everything contributes 0
  }
  // limits are checked before anything is enqueued or allocated (outputs/plan untouched on error)
  unsigned bpr = 0;
  if (p->mtab) {
    const unsigned outs = (unsigned)p->w_max * sftk::TAB_R * (sftk::TAB_Q + 1);
    bpr = (outs + 255) / 256;
    if (bpr < 1) bpr = 1;
    if ((double)bpr * (double)N > 2.0e9) return fail(p, SFT_EUNSUPPORTED, "moment-table build grid too large");
  }
  const float2 *d_raw = nullptr;
  const double *d_scale = nullptr, *d_shape = nullptr;
  void *tmp = nullptr;
  // from here on the channel's tables are being replaced: a failure leaves the channel unloaded
  p->loaded[channel] = false;
  cudaError_t e = cudaSuccess;
  auto ok = [&](cudaError_t r) { if (e == cudaSuccess && r != cudaSuccess) e = r; return e == cudaSuccess; };
  if (mem == SFT_MEM_HOST) {
    const size_t b_raw = N * nb * sizeof(float2), b_scale = N * sizeof(double), b_shape = psd_shape ? nb * sizeof(double) : 0;
    const size_t o_scale = (b_raw + 255) & ~size_t(255), o_shape = (o_scale + b_scale + 255) & ~size_t(255);
    cudaError_t ea = cudaMalloc(&tmp, o_shape + b_shape + 256);
    if (ea != cudaSuccess) return fail(p, SFT_ENOMEM, "cudaMalloc staging: %s", cudaGetErrorString(ea));
    char *base = (char *)tmp;
    ok(cudaMemcpyAsync(base, sft_bins, b_raw, cudaMemcpyHostToDevice, p->stream));
    ok(cudaMemcpyAsync(base + o_scale, psd_scale, b_scale, cudaMemcpyHostToDevice, p->stream));
    if (psd_shape) ok(cudaMemcpyAsync(base + o_shape, psd_shape, b_shape, cudaMemcpyHostToDevice, p->stream));
    if (p->d.response == SFT_RESP_TABLE)
      ok(cudaMemcpyAsync(p->rtab + (size_t)channel * N, response, N * sizeof(float2), cudaMemcpyHostToDevice, p->stream));
    d_raw = (const float2 *)base;
    d_scale = (const double *)(base + o_scale);
    d_shape = psd_shape ? (const double *)(base + o_shape) : nullptr;
  } else {
    d_raw = (const float2 *)sft_bins;
    d_scale = psd_scale;
    d_shape = psd_shape;
    if (p->d.response == SFT_RESP_TABLE)
      ok(cudaMemcpyAsync(p->rtab + (size_t)channel * N, response, N * sizeof(float2), cudaMemcpyDeviceToDevice, p->stream));
  }
  const size_t C = p->d.n_channels, npair = p->npair;
  if (e == cudaSuccess) {
    sftk::sft_whiten_kernel<<<(unsigned)N, 128, 0, p->stream>>>(
        d_raw, d_scale, d_shape, (int)N, (int)nb, p->d.k_lo, p->kv_lo, p->kv_hi, p->PAD, p->npair, p->d.t_sft, S_ref,
        p->Dp + (size_t)channel * N * npair, p->Dp + (C + (size_t)channel) * N * npair, p->us2 + (size_t)channel * N);
    sftk::sft_ub2_kernel<<<(unsigned)((2 * npair + 255) / 256), 256, 0, p->stream>>>(
        d_shape, (int)nb, p->d.k_lo, p->kv_lo, p->kv_hi, p->PAD, p->npair, S_ref, p->ubp + (size_t)channel * npair,
        p->ubp + (C + (size_t)channel) * npair);
    p->launches += 2;
    if (d_shape) ok(cudaMemcpyAsync(p->shape_dev + (size_t)channel * nb, d_shape, nb * sizeof(double), cudaMemcpyDeviceToDevice, p->stream));
    if (p->mtab) {
      sftk::sft_mtab_kernel<<<(unsigned)(bpr * N), 256, 0, p->stream>>>(
          p->Dp + (size_t)channel * N * npair, p->npair, p->tblk, 0, p->d.K, p->ptab, bpr, (float2 *)(p->mtab + (size_t)channel * p->m_f4_chan));
      sftk::sft_htab_kernel<<<(unsigned)(p->n_kc * sftk::HTAB_R), 64, 0, p->stream>>>(
          p->ubp + (size_t)channel * npair, p->d.K, (float *)(p->htab + (size_t)channel * p->n_kc * sftk::HTAB_R * (sftk::HTAB_W / 4)));
      sftk::sft_htab1_kernel<<<(unsigned)(p->n_kc * sftk::HT1_R), 64, 0, p->stream>>>(
          p->ubp + (size_t)channel * npair, p->d.K, p->htab1 + (size_t)channel * p->n_kc * sftk::HT1_R);
      p->launches += 3;
    }
    ok(cudaGetLastError());
  }
  // the staging buffer and the caller's host arrays may be in flight: always drain the stream before returning
  cudaError_t e2 = cudaStreamSynchronize(p->stream);
  if (tmp) cudaFree(tmp);
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "sft_load_data (copy/launch): %s", cudaGetErrorString(e));
  if (e2 != cudaSuccess) return fail(p, SFT_ECUDA, "sft_load_data: %s", cudaGetErrorString(e2));
  p->sigma[channel] = sqrt(p->d.t_sft / S_ref);
  p->s_ref[channel] = S_ref;
  p->has_shape[channel] = psd_shape != nullptr;
  p->loaded[channel] = true;
  return SFT_OK;
}

// Streaming (section V.A: SFTs "can be computed online and in parallel as data arrives"): replaces the SFT slots
// [first_sft, first_sft + n_new) of a loaded channel - whitening with the channel's PSD shape, the rows of the pair-planar
// store and of the moment table - in place; nothing else of the plan is touched or rebuilt.
SFT_API sft_status sft_append_sfts(sft_plan *p, int32_t channel, int64_t first_sft, int64_t n_new, const float *sft_bins,
                                   const double *psd_scale, const float *response, int32_t mem) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (channel < 0 || channel >= p->d.n_channels) return fail(p, SFT_EINVAL, "channel %d outside 0..%d", channel, p->d.n_channels - 1);
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(p, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  if (n_new < 0 || first_sft < 0 || first_sft + n_new > p->d.n_sft)
    return fail(p, SFT_ESHAPE, "slots [%lld, %lld) outside the plan's %lld SFT slots", (long long)first_sft, (long long)(first_sft + n_new),
                (long long)p->d.n_sft);
  if (!p->loaded[channel]) return fail(p, SFT_ENODATA, "channel %d has no data yet: sft_load_data fixes its PSD shape first", channel);
  if (n_new == 0) return SFT_OK;
  if (!sft_bins || !psd_scale) return fail(p, SFT_EINVAL, "sft_bins and psd_scale are required");
  if (p->d.response == SFT_RESP_TABLE && !response) return fail(p, SFT_EINVAL, "response table required by SFT_RESP_TABLE");
  CU(p, cudaSetDevice(p->d.device));
  const size_t N = p->d.n_sft, nb = p->nb, nn = (size_t)n_new, a0 = (size_t)first_sft, C = p->d.n_channels, npair = p->npair;
  unsigned bpr = 0;
  if (p->mtab) {
    bpr = ((unsigned)p->w_max * sftk::TAB_R * (sftk::TAB_Q + 1) + 255) / 256;
    if (bpr < 1) bpr = 1;
    if ((double)bpr * (double)nn > 2.0e9) return fail(p, SFT_EUNSUPPORTED, "moment-table build grid too large");
  }
  const float2 *d_raw = (const float2 *)sft_bins;
  const double *d_scale = psd_scale;
  void *tmp = nullptr;
  cudaError_t e = cudaSuccess;
  auto ok = [&](cudaError_t r) { if (e == cudaSuccess && r != cudaSuccess) e = r; return e == cudaSuccess; };
  if (mem == SFT_MEM_HOST) {
    const size_t b_raw = nn * nb * sizeof(float2), o_scale = (b_raw + 255) & ~size_t(255);
    cudaError_t ea = cudaMalloc(&tmp, o_scale + nn * sizeof(double) + 256);
    if (ea != cudaSuccess) return fail(p, SFT_ENOMEM, "cudaMalloc staging: %s", cudaGetErrorString(ea));
    ok(cudaMemcpyAsync(tmp, sft_bins, b_raw, cudaMemcpyHostToDevice, p->stream));
    ok(cudaMemcpyAsync((char *)tmp + o_scale, psd_scale, nn * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    d_raw = (const float2 *)tmp;
    d_scale = (const double *)((char *)tmp + o_scale);
  }
  if (p->d.response == SFT_RESP_TABLE)
    ok(cudaMemcpyAsync(p->rtab + (size_t)channel * N + a0, response, nn * sizeof(float2),
                       mem == SFT_MEM_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, p->stream));
  if (e == cudaSuccess) {
    const double *d_shape = p->has_shape[channel] ? p->shape_dev + (size_t)channel * nb : nullptr;
    float4 *D0 = p->Dp + ((size_t)channel * N + a0) * npair, *D1 = p->Dp + ((C + (size_t)channel) * N + a0) * npair;
    sftk::sft_whiten_kernel<<<(unsigned)nn, 128, 0, p->stream>>>(d_raw, d_scale, d_shape, (int)nn, (int)nb, p->d.k_lo, p->kv_lo, p->kv_hi,
                                                                 p->PAD, p->npair, p->d.t_sft, p->s_ref[channel], D0, D1,
                                                                 p->us2 + (size_t)channel * N + a0);
    p->launches++;
    if (p->mtab) {
      sftk::sft_mtab_kernel<<<(unsigned)(bpr * nn), 256, 0, p->stream>>>(D0, p->npair, p->tblk, (int)a0, p->d.K, p->ptab, bpr,
                                                                        (float2 *)(p->mtab + (size_t)channel * p->m_f4_chan));
      p->launches++;
    }
    ok(cudaGetLastError());
  }
  cudaError_t e2 = (tmp || e != cudaSuccess) ? cudaStreamSynchronize(p->stream) : cudaSuccess;   // host staging in flight
  if (tmp) cudaFree(tmp);
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "sft_append_sfts (copy/launch): %s", cudaGetErrorString(e));
  if (e2 != cudaSuccess) return fail(p, SFT_ECUDA, "sft_append_sfts: %s", cudaGetErrorString(e2));
  return SFT_OK;
}

// ---------------------------------------------------------------------------------------------
// Data SFTs from the time series (sft_ingest.cuh).  `x` and `bins` are DEVICE pointers here.
static cudaError_t compute_sfts_device(cudaStream_t stream, const double *x, int64_t n_sft, int n, double dt, int k_lo,
                                       int k_hi, float2 *bins, long long *launches) {
  const int nb = k_hi - k_lo;
  const bool pow2 = n >= 64 && n <= sftk::FFT_MAX_N && (n & (n - 1)) == 0 && (((size_t)x & 15) == 0);
  if (pow2) {
    // twiddle tables are kept per (device, n) for the life of the process (<= 64 KB each)
    static std::mutex mu;
    static std::vector<std::pair<std::pair<int, int>, float2 *>> cache;
    int dev = 0;
    cudaGetDevice(&dev);
    float2 *W = nullptr;
    {
      std::lock_guard<std::mutex> lk(mu);
      for (auto &c : cache)
        if (c.first.first == dev && c.first.second == n) W = c.second;
      if (!W) {
        cudaError_t e = cudaMalloc((void **)&W, (size_t)(n / 2) * sizeof(float2));
        if (e != cudaSuccess) return e;
        sftk::sft_twiddle_kernel<<<(n / 2 + 255) / 256, 256, 0, stream>>>(n, W);
        e = cudaStreamSynchronize(stream);
        if (e != cudaSuccess) { cudaFree(W); return e; }
        cache.push_back({{dev, n}, W});
        if (launches) *launches += 1;
      }
    }
    int log2m = 0;
    while ((1 << log2m) < n / 2) ++log2m;
    int n_sm = 1;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    auto launch = [&](auto kernel, size_t smem, auto... args) {
      cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      int per_sm = 1;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, 256, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
      long long grid = (long long)n_sm * per_sm;
      if (grid > n_sft) grid = n_sft;
      kernel<<<(unsigned)grid, 256, smem, stream>>>(args...);
    };
    auto launch_lb = [&](auto kernel, size_t smem, auto... args) {
      cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      int per_sm = 1;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, 256, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
      // persistent blocks, prefetch distance = one round of the grid (one block per segment measured 4 % slower)
      const long long resident = (long long)n_sm * per_sm, grid = resident < n_sft ? resident : n_sft;
      kernel<<<(unsigned)grid, 256, smem, stream>>>(args..., (int)grid);
    };
    const size_t smem = (size_t)(n / 2 + n / 32 + 1) * sizeof(float2);
    // a band of at most 256 bins inside [1, n/2]: output-pruned transform (two radix-16 passes, then one sum per output).
    // SFT_INGEST_FULL_FFT in the environment forces the full transform (measurement switch, profiles/r02_ingest.md).
    const bool narrow = nb <= 256 && k_lo >= 1 && k_hi <= n / 2 && log2m >= 11 && log2m <= 13 && !getenv("SFT_INGEST_FULL_FFT");
    if (narrow && log2m == 13)
      launch_lb(sftk::sft_rfft_lowband_kernel<5>, smem + 20 * 32 * sizeof(float2), x, (int)n_sft, dt, k_lo, nb, (const float2 *)W, bins);
    else if (narrow && log2m == 12)
      launch_lb(sftk::sft_rfft_lowband_kernel<4>, smem + 20 * 16 * sizeof(float2), x, (int)n_sft, dt, k_lo, nb, (const float2 *)W, bins);
    else if (narrow)
      launch_lb(sftk::sft_rfft_lowband_kernel<3>, smem + 20 * 8 * sizeof(float2), x, (int)n_sft, dt, k_lo, nb, (const float2 *)W, bins);
    else
      launch(sftk::sft_rfft_band_kernel, smem, x, (int)n_sft, n, log2m, dt, k_lo, nb, (const float2 *)W, bins);
    if (launches) *launches += 1;
    return cudaGetLastError();
  }
  sftk::sft_dft_band_kernel<<<(unsigned)n_sft, 256, 0, stream>>>(x, n, dt, k_lo, nb, bins);
  if (launches) *launches += 1;
  return cudaGetLastError();
}

SFT_API sft_status sft_compute_sfts(int32_t device, void *stream, const double *x, int64_t n_sft, int32_t n, double dt,
                                    int32_t k_lo, int32_t k_hi, float *bins, int32_t mem) {
  g_create_err[0] = 0;
  if (!x || !bins) return fail(nullptr, SFT_EINVAL, "sft_compute_sfts: x and bins are required");
  if (n_sft < 1 || n_sft > (1ll << 30) || n < 2 || !(dt > 0.0) || k_lo < 0 || k_hi <= k_lo)
    return fail(nullptr, SFT_EINVAL, "sft_compute_sfts: need n_sft >= 1, n >= 2, dt > 0, 0 <= k_lo < k_hi");
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(nullptr, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  CU(nullptr, cudaSetDevice(device));
  cudaStream_t st = (cudaStream_t)stream;
  const size_t nb = (size_t)(k_hi - k_lo), b_x = (size_t)n_sft * n * sizeof(double), b_out = (size_t)n_sft * nb * sizeof(float2);
  const double *d_x = x;
  float2 *d_out = (float2 *)bins;
  void *tmp = nullptr;
  if (mem == SFT_MEM_HOST) {
    cudaError_t e = cudaMalloc(&tmp, b_x + b_out + 256);
    if (e != cudaSuccess) return fail(nullptr, SFT_ENOMEM, "cudaMalloc staging: %s", cudaGetErrorString(e));
    cudaError_t ec = cudaMemcpyAsync(tmp, x, b_x, cudaMemcpyHostToDevice, st);
    if (ec != cudaSuccess) { cudaStreamSynchronize(st); cudaFree(tmp); return fail(nullptr, SFT_ECUDA, "sft_compute_sfts: %s", cudaGetErrorString(ec)); }
    d_x = (const double *)tmp;
    d_out = (float2 *)((char *)tmp + ((b_x + 255) & ~size_t(255)));
  }
  cudaError_t e = compute_sfts_device(st, d_x, n_sft, n, dt, k_lo, k_hi, d_out, nullptr);
  if (e == cudaSuccess && mem == SFT_MEM_HOST) e = cudaMemcpyAsync(bins, d_out, b_out, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (tmp) { cudaStreamSynchronize(st); cudaFree(tmp); }
  if (e != cudaSuccess) return fail(nullptr, SFT_ECUDA, "sft_compute_sfts: %s", cudaGetErrorString(e));
  return SFT_OK;
}

// Per-SFT noise level from the data (sft_ingest.cuh).  Device pointers.
static cudaError_t estimate_scale_device(cudaStream_t st, const float2 *bins, int64_t n_sft, int nb, const double *shape, double T,
                                         int k_lo, int n_samp, int w, double *scale, unsigned char *flag, int pool_max) {
  int npow2 = 1;
  while (npow2 < pool_max) npow2 <<= 1;
  sftk::sft_nonzero_kernel<<<(unsigned)n_sft, 128, 0, st>>>(bins, nb, flag);
  sftk::sft_psd_scale_kernel<<<(unsigned)n_sft, 256, (size_t)npow2 * sizeof(float), st>>>(bins, flag, shape, (int)n_sft, nb, k_lo, n_samp,
                                                                                          0.5 * T, w, npow2, scale);
  return cudaGetLastError();
}

SFT_API sft_status sft_estimate_psd_scale(int32_t device, void *stream, const float *sft_bins, int64_t n_sft, int32_t k_lo,
                                          int32_t k_hi, int32_t n_samp, double t_sft, const double *psd_shape, int32_t half_window,
                                          double *psd_scale, int32_t mem) {
  g_create_err[0] = 0;
  if (!sft_bins || !psd_scale) return fail(nullptr, SFT_EINVAL, "sft_estimate_psd_scale: sft_bins and psd_scale are required");
  if (n_sft < 1 || n_sft > (1ll << 30) || k_lo < 0 || k_hi <= k_lo || n_samp < 2 || !(t_sft > 0.0) || half_window < 0)
    return fail(nullptr, SFT_EINVAL, "sft_estimate_psd_scale: need n_sft >= 1, 0 <= k_lo < k_hi, n_samp >= 2, t_sft > 0, half_window >= 0");
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(nullptr, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  const int nb = k_hi - k_lo;
  const int q0 = k_lo < 1 ? 1 - k_lo : 0, q1 = nb < n_samp / 2 - k_lo ? nb : n_samp / 2 - k_lo;
  const long long pool = (long long)(2 * half_window + 1) * (q1 > q0 ? q1 - q0 : 0);
  if (pool > sftk::PSD_MAX_VALUES)
    return fail(nullptr, SFT_EUNSUPPORTED, "pool of %lld values per SFT exceeds %d: use a smaller half_window or band", pool, sftk::PSD_MAX_VALUES);
  CU(nullptr, cudaSetDevice(device));
  cudaStream_t st = (cudaStream_t)stream;
  const size_t b_bins = (size_t)n_sft * nb * sizeof(float2), b_shape = psd_shape ? nb * sizeof(double) : 0, b_scale = (size_t)n_sft * sizeof(double);
  void *tmp = nullptr;
  const size_t o_shape = (b_bins + 255) & ~size_t(255), o_scale = (o_shape + b_shape + 255) & ~size_t(255), o_flag = o_scale + b_scale;
  cudaError_t e = cudaMalloc(&tmp, (mem == SFT_MEM_HOST ? o_flag : 0) + (size_t)n_sft + 512);
  if (e != cudaSuccess) return fail(nullptr, SFT_ENOMEM, "cudaMalloc staging: %s", cudaGetErrorString(e));
  const float2 *d_bins = (const float2 *)sft_bins;
  const double *d_shape = psd_shape;
  double *d_scale = psd_scale;
  unsigned char *d_flag = (unsigned char *)tmp;
  if (mem == SFT_MEM_HOST) {
    char *base = (char *)tmp;
    e = cudaMemcpyAsync(base, sft_bins, b_bins, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && psd_shape) e = cudaMemcpyAsync(base + o_shape, psd_shape, b_shape, cudaMemcpyHostToDevice, st);
    d_bins = (const float2 *)base;
    d_shape = psd_shape ? (const double *)(base + o_shape) : nullptr;
    d_scale = (double *)(base + o_scale);
    d_flag = (unsigned char *)(base + o_flag);
  }
  if (e == cudaSuccess) e = estimate_scale_device(st, d_bins, n_sft, nb, d_shape, t_sft, k_lo, n_samp, half_window, d_scale, d_flag, (int)(pool > 1 ? pool : 1));
  if (e == cudaSuccess && mem == SFT_MEM_HOST) e = cudaMemcpyAsync(psd_scale, d_scale, b_scale, cudaMemcpyDeviceToHost, st);
  cudaError_t e2 = cudaStreamSynchronize(st);
  cudaFree(tmp);
  if (e != cudaSuccess || e2 != cudaSuccess) return fail(nullptr, SFT_ECUDA, "sft_estimate_psd_scale: %s", cudaGetErrorString(e != cudaSuccess ? e : e2));
  return SFT_OK;
}

SFT_API sft_status sft_ingest_timeseries(sft_plan *p, int32_t channel, const double *x, int64_t n_samples,
                                         const double *psd_scale, const double *psd_shape, const float *response, int32_t mem) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (!x) return fail(p, SFT_EINVAL, "x is required");
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(p, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  const size_t N = p->d.n_sft, n = p->n_samp, nb = p->nb;
  if (!psd_scale) {                      // estimated from the data: one median over the band per SFT (sft_estimate_psd_scale)
    const long long pool = (long long)p->kv_hi - p->kv_lo;
    if (pool > sftk::PSD_MAX_VALUES) return fail(p, SFT_EUNSUPPORTED, "psd_scale = NULL: the band holds more than %d bins", sftk::PSD_MAX_VALUES);
  }
  if (n_samples < (int64_t)(N * n)) return fail(p, SFT_ESHAPE, "%lld samples < n_sft * n = %zu", (long long)n_samples, N * n);
  CU(p, cudaSetDevice(p->d.device));
  const size_t b_x = N * n * sizeof(double), b_bins = N * nb * sizeof(float2);
  void *tmp = nullptr;
  cudaError_t e = cudaMalloc(&tmp, (mem == SFT_MEM_HOST ? b_x : 0) + b_bins + 512);
  if (e != cudaSuccess) return fail(p, SFT_ENOMEM, "cudaMalloc staging: %s", cudaGetErrorString(e));
  float2 *d_bins = (float2 *)tmp;
  const double *d_x = x;
  if (mem == SFT_MEM_HOST) {
    double *dx = (double *)((char *)tmp + ((b_bins + 255) & ~size_t(255)));
    e = cudaMemcpyAsync(dx, x, b_x, cudaMemcpyHostToDevice, p->stream);
    if (e != cudaSuccess) { cudaStreamSynchronize(p->stream); cudaFree(tmp); return fail(p, SFT_ECUDA, "series copy: %s", cudaGetErrorString(e)); }
    d_x = dx;
  }
  e = compute_sfts_device(p->stream, d_x, (int64_t)N, (int)n, 1.0 / p->d.fs, p->d.k_lo, p->d.k_hi, d_bins, &p->launches);
  if (e != cudaSuccess) { cudaStreamSynchronize(p->stream); cudaFree(tmp); return fail(p, SFT_ECUDA, "SFT kernel: %s", cudaGetErrorString(e)); }
  // the noise description may live on either side: bring it to the device, then the common whitening path
  sft_status st = SFT_OK;
  void *tmp2 = nullptr;
  const double *d_scale = psd_scale, *d_shape = psd_shape;
  const float *d_resp = response;
  if (mem == SFT_MEM_HOST || !psd_scale) {
    const bool host = mem == SFT_MEM_HOST;
    const size_t b_scale = N * sizeof(double), b_shape = (psd_shape && host) ? nb * sizeof(double) : 0;
    const size_t b_resp = (response && host && p->d.response == SFT_RESP_TABLE) ? N * sizeof(float2) : 0;
    e = cudaMalloc(&tmp2, b_scale + b_shape + b_resp + N + 1024);
    if (e != cudaSuccess) { cudaStreamSynchronize(p->stream); cudaFree(tmp); return fail(p, SFT_ENOMEM, "cudaMalloc staging: %s", cudaGetErrorString(e)); }
    char *q = (char *)tmp2;
    e = psd_scale && host ? cudaMemcpyAsync(q, psd_scale, b_scale, cudaMemcpyHostToDevice, p->stream) : cudaSuccess;
    if (!psd_scale || host) d_scale = (const double *)q;
    double *est = (double *)q;
    q += (b_scale + 255) & ~size_t(255);
    if (psd_shape && e == cudaSuccess) { e = cudaMemcpyAsync(q, psd_shape, b_shape, cudaMemcpyHostToDevice, p->stream); d_shape = (const double *)q; q += (b_shape + 255) & ~size_t(255); }
    if (b_resp && e == cudaSuccess) { e = cudaMemcpyAsync(q, response, b_resp, cudaMemcpyHostToDevice, p->stream); d_resp = (const float *)q; q += (b_resp + 255) & ~size_t(255); }
    if (!psd_scale && e == cudaSuccess) {
      e = estimate_scale_device(p->stream, d_bins, (int64_t)N, (int)nb, d_shape, p->d.t_sft, p->d.k_lo, p->n_samp, 0, est, (unsigned char *)q,
                                p->kv_hi > p->kv_lo ? p->kv_hi - p->kv_lo : 1);
      p->launches += 2;
    }
    if (e != cudaSuccess) {
      cudaStreamSynchronize(p->stream); cudaFree(tmp); cudaFree(tmp2);
      return fail(p, SFT_ECUDA, "noise-description copy: %s", cudaGetErrorString(e));
    }
  }
  st = sft_load_data(p, channel, (const float *)d_bins, d_scale, d_shape, d_resp, SFT_MEM_DEVICE);
  cudaStreamSynchronize(p->stream);
  cudaFree(tmp);
  if (tmp2) cudaFree(tmp2);
  return st;
}

// ---------------------------------------------------------------------------------------------
static void fill_kparams(const sft_plan *p, KParams &k) {
  memset(&k, 0, sizeof(k));
  k.C = p->d.n_channels;
  k.n_sft = (int)p->d.n_sft;
  k.nb = p->nb;
  k.k_lo = p->d.k_lo;
  k.kv_lo = p->kv_lo;
  k.kv_hi = p->kv_hi;
  k.K = p->d.K;
  k.PAD = p->PAD;
  k.npair = p->npair;
  k.kwin0 = p->d.k_lo + p->d.K - p->PAD;
  k.jmax = p->nb - 1 + p->PAD - 2;
  k.dstride = (unsigned)(p->d.n_sft * p->npair);
  k.cstrideD = (unsigned)(p->d.n_channels * p->d.n_sft * p->npair);
  k.cstrideU = (unsigned)(p->d.n_channels * p->npair);
  k.kernel = p->d.kernel;
  k.pn1 = p->d.waveform;                          // PN order code: 0, 1 (1PN), 2 (1.5PN)
  k.response = p->d.response;
  k.phase_path = p->d.phase_path;
  k.T = p->d.t_sft;
  k.t0 = p->d.t0;
  k.f_loT = p->d.f_lo * p->d.t_sft;
  k.f_hiT = fmin(p->d.f_hi * p->d.t_sft, 1.0e9);   // keeps k_c inside int32 (bins beyond 1e9 do not exist)
  k.inv_fref = 1.0 / p->d.f_ref;
  for (int c = 0; c < SFT_MAX_CHANNELS; ++c) {
    k.sigma[c] = p->sigma[c];
    k.chi[c] = p->d.resp_chi[c];
  }
  k.depth = (float)p->d.resp_depth;
  k.mtab = p->mtab;
  k.htab = p->htab;
  k.htab1 = p->htab1;
  k.h1chan = (unsigned)(p->n_kc * sftk::HT1_R);
  k.tblk = p->tblk;
  k.banded = p->banded ? 1 : 0;
  k.mrow0 = (unsigned)p->n_node * (unsigned)((sftk::TAB_Q + 1) / 2);
  k.mchan = p->mtab ? (unsigned)p->m_f4_chan : 0u;
  k.hchan = (unsigned)(p->n_kc * sftk::HTAB_R * (sftk::HTAB_W / 4));
  k.b_table = p->mtab ? sftk::B_TABLE : -1.0f;
  k.b_table2 = p->mtab ? sftk::B_TABLE2 : -1.0f;
  k.Dp = p->Dp;
  k.ubp = p->ubp;
  k.us2 = p->us2;
  k.rtab = p->rtab;
#ifdef SFT_CHECKED
  {                                                    // extents of the allocations (sft_plan_create, table_layout), in entries
    const unsigned long long C = p->d.n_channels, N = p->d.n_sft;
    k.chk = p->chk;
    k.n_Dp = (2 * C * N + 1) * (unsigned long long)p->npair;
    k.n_ubp = 2 * C * (unsigned long long)p->npair;
    k.n_sl = C * N;
    k.n_mtab = p->mtab ? C * (unsigned long long)p->m_f4_chan : 0;
    k.n_htab = p->htab ? C * (unsigned long long)p->n_kc * sftk::HTAB_R * (sftk::HTAB_W / 4) : 0;
    k.n_htab1 = p->htab1 ? C * (unsigned long long)p->n_kc * sftk::HT1_R : 0;
    k.n_tblk = p->tblk ? (N + 31) / 32 : 0;
  }
#endif
}

// The variants of the fused main kernel live in sft_var_*.cu (sft_launch.cuh): ask the units in turn.
static cudaError_t launch_main(sft_plan *p, const KParams &k, int mode) {
  cudaEventRecord(p->ev0, p->stream);             // (the work-unit counter was zeroed by sft_tmpl_kernel)
  const bool diag = k.kc_out != nullptr || k.path_counts != nullptr || k.phase_path != 0;
  sftl::Key key;
  key.mode = mode;
  key.C = k.C;
  key.K = k.K;
  key.bns32 = mode != 2 && k.kc_out == nullptr && k.path_counts == nullptr && k.phase_path == 1 && k.kernel == 1 && k.pn1 == 1 &&
              k.response == 0 && k.C == 1 && k.K == 8;
  key.bns = !diag && k.kernel == 1 && k.pn1 == 1 && k.response == 0;
  key.newt = !diag && k.kernel == 1 && k.pn1 == 0 && k.response == 0;
  key.lisa = !diag && k.kernel == 1 && k.pn1 == 1 && k.response == 2;
  const sftl::Ctx ctx = {p->stream, p->n_sm, p->banded};
  const bool done = sftl::launch_bns(key, ctx, k) || sftl::launch_misc(key, ctx, k) || sftl::launch_lisa(key, ctx, k) ||
                    sftl::launch_any1(key, ctx, k) || sftl::launch_any2(key, ctx, k) || sftl::launch_any3(key, ctx, k) ||
                    sftl::launch_any4(key, ctx, k);
  cudaEventRecord(p->ev1, p->stream);
  p->timed = true;
  p->launches++;
#ifdef SFT_CHECKED
  if (done) {                                          // the site (sftk::ChkSite) of the first failed bounds check, if any
    unsigned site = 0;
    cudaError_t ec = cudaStreamSynchronize(p->stream);
    if (ec == cudaSuccess) ec = cudaMemcpy(&site, p->chk, sizeof(site), cudaMemcpyDeviceToHost);
    if (ec != cudaSuccess) return ec;
    if (site != 0) {
      fprintf(stderr, "sft_b200 (checked build): bounds check failed at site %u (sftk::ChkSite)\n", site);
      cudaMemset(p->chk, 0, sizeof(unsigned));
      return cudaErrorAssert;
    }
  }
#endif
  return done ? cudaGetLastError() : cudaErrorInvalidConfiguration;
}

static sft_status prepare(sft_plan *p, int64_t nT, const double *params, int32_t mem, KParams &k, bool cumulative, int nq = 3) {
  for (int c = 0; c < p->d.n_channels; ++c)
    if (!p->loaded[c]) return fail(p, SFT_ENODATA, "channel %d has no data (call sft_load_data)", c);
  if (nT > (1ll << 31) - 1) return fail(p, SFT_EINVAL, "n_templates too large");
  if (cumulative && (double)nT * (double)p->d.n_sft > 4.0e10) return fail(p, SFT_EINVAL, "cumulative output too large");
  CU(p, cudaSetDevice(p->d.device));
  fill_kparams(p, k);
  k.nT = nT;
  // SFTs per work unit: enough units (>= ~16 per resident warp) for the dynamic scheduler to balance,
  // but no more chunks than that (the chunk totals cost 24 bytes per template and chunk)
  k.n_tgroups = (int)((nT + 31) / 32);
  int chunk = p->chunk_user;
  if (chunk <= 0) {
    const long long target_units = 16ll * p->n_sm * 24;
    long long want_chunks = (target_units + k.n_tgroups - 1) / k.n_tgroups;
    if (want_chunks < 1) want_chunks = 1;
    chunk = (int)((k.n_sft + want_chunks - 1) / want_chunks);
    if (chunk < 32) chunk = 32;
    chunk = ((chunk + 31) / 32) * 32;            // work units aligned to the blocks of 32 SFT slots of the fast path / table layout
  }
  if (cumulative) chunk = sftk::SUB;          // single-pass scan: one work unit = one block of 32 SFT slots (scan_store)
  if (chunk > k.n_sft && !cumulative) chunk = k.n_sft;
  k.chunk = chunk;
  k.n_chunks = (k.n_sft + chunk - 1) / chunk;
  sft_status st = SFT_OK;
  if (cumulative) {
    // look-back records: per (unit, template) two 16-byte words {xh, hh} (aggregate, inclusive), each carrying the 16-bit tag
    // of the call that wrote it (scan_publish), so nothing is cleared between calls; a fresh or regrown buffer is zeroed (tag 0
    // is never used) and so is the buffer when the tag wraps.
    const size_t ent = (size_t)k.n_chunks * (size_t)nT, need = ent * 2 * sizeof(double2);
    if (p->scan_bytes < need || p->epoch >= 0xfffeu) {
      st = grow(p, &p->scan, &p->scan_bytes, need);
      if (st != SFT_OK) return st;
      CU(p, cudaMemsetAsync(p->scan, 0, p->scan_bytes, p->stream));
      p->epoch = 0;
    }
    p->epoch++;
    k.scanA = (double2 *)p->scan;
    k.scanP = k.scanA + ent;
    k.epoch = p->epoch;
#ifdef SFT_CHECKED
    k.n_scan = ent;
#endif
  } else {
    st = grow(p, (void **)&p->part, &p->part_bytes, (size_t)k.n_chunks * nq * nT * sizeof(double));
    if (st != SFT_OK) return st;
    k.part = p->part;
#ifdef SFT_CHECKED
    k.n_part = (unsigned long long)k.n_chunks * nq * nT;
#endif
  }
  if ((double)k.n_tgroups * (double)k.n_chunks > 2.0e9) return fail(p, SFT_EINVAL, "too many work units: raise sfts_per_block");
  k.n_items = k.n_tgroups * k.n_chunks;
  k.counter = p->counter;
  st = grow(p, (void **)&p->td, &p->td_bytes, (size_t)sftk::TD_N * nT * sizeof(double));
  if (st != SFT_OK) return st;
  st = grow(p, (void **)&p->tf, &p->tf_bytes, (size_t)sftk::TF_N * nT * sizeof(float));
  if (st != SFT_OK) return st;
  k.td = p->td;
  k.tf = p->tf;
  if (mem == SFT_MEM_HOST) {
    st = grow(p, (void **)&p->d_params, &p->params_bytes, (size_t)nT * SFT_NPARAM * sizeof(double));
    if (st != SFT_OK) return st;
    CU(p, cudaMemcpyAsync(p->d_params, params, (size_t)nT * SFT_NPARAM * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    k.params = p->d_params;
  } else {
    k.params = params;
  }
  sftk::sft_tmpl_kernel<<<(unsigned)((nT + 127) / 128), 128, 0, p->stream>>>(k, p->td, p->tf);
  p->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "template kernel launch: %s", cudaGetErrorString(e));
  return SFT_OK;
}

SFT_API sft_status sft_inner_products(sft_plan *p, int64_t nT, const double *params, double *xh, double *hh,
                                         double *xh_im, int32_t *kc_out, int32_t mem) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (nT < 0) return fail(p, SFT_EINVAL, "n_templates < 0");
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(p, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  if (nT == 0) return SFT_OK;
  if (!params || !xh || !hh) return fail(p, SFT_EINVAL, "params, xh and hh are required");
  KParams k;
  sft_status st = prepare(p, nT, params, mem, k, false);
  if (st != SFT_OK) return st;
  const size_t C = p->d.n_channels, N = p->d.n_sft;
  double *d_xh = xh, *d_hh = hh, *d_xi = xh_im;
  int *d_kc = kc_out;
  if (mem == SFT_MEM_HOST) {
    const size_t b_vec = (size_t)nT * sizeof(double);
    const size_t b_kc = kc_out ? (size_t)nT * C * N * sizeof(int) : 0;
    st = grow(p, &p->d_out, &p->out_bytes, 3 * b_vec + b_kc + 256);
    if (st != SFT_OK) return st;
    d_xh = (double *)p->d_out;
    d_hh = d_xh + nT;
    d_xi = d_hh + nT;
    d_kc = kc_out ? (int *)(d_xi + nT) : nullptr;
  }
  k.kc_out = d_kc;
#ifdef SFT_CHECKED
  k.n_kc = d_kc ? (unsigned long long)nT * C * N : 0;
#endif
  k.path_counts = d_kc ? p->path_counts : nullptr;     // the diagnostic call also counts the evaluator paths
  if (d_kc) CU(p, cudaMemsetAsync(p->path_counts, 0, sftk::PATH_N * sizeof(unsigned long long), p->stream));
  cudaError_t e = launch_main(p, k, 0);
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "main kernel launch: %s", cudaGetErrorString(e));
  sftk::RedOut ro = {{d_xh, d_hh, d_xi, nullptr, nullptr, nullptr, nullptr}};
  sftk::sft_reduce_kernel<<<dim3((unsigned)((nT + 31) / 32), 3), 32 * sftk::RED_SLICES, 0, p->stream>>>(p->part, nT, k.n_chunks, 3, ro);
  p->launches++;
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "reduce kernel launch: %s", cudaGetErrorString(e));
  if (mem == SFT_MEM_HOST) {
    // results go to caller memory only after the stream finished without error
    st = grow_pinned(p, 3 * (size_t)nT * sizeof(double));
    if (st != SFT_OK) return st;
    double *h = (double *)p->h_pin;
    CU(p, cudaMemcpyAsync(h, d_xh, 3 * (size_t)nT * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    memcpy(xh, h, (size_t)nT * sizeof(double));
    memcpy(hh, h + nT, (size_t)nT * sizeof(double));
    if (xh_im) memcpy(xh_im, h + 2 * nT, (size_t)nT * sizeof(double));
    if (kc_out) {
      CU(p, cudaMemcpyAsync(kc_out, d_kc, (size_t)nT * C * N * sizeof(int), cudaMemcpyDeviceToHost, p->stream));
      CU(p, cudaStreamSynchronize(p->stream));
    }
  }
  return SFT_OK;
}

SFT_API sft_status sft_statistics(sft_plan *p, int64_t nT, const double *xh, const double *xh_im, const double *hh,
                                  double *loglike, double *rho2_phase_max, int32_t mem) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (nT < 0) return fail(p, SFT_EINVAL, "n_templates < 0");
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(p, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  if (nT == 0) return SFT_OK;
  if (!xh || !xh_im || !hh) return fail(p, SFT_EINVAL, "xh, xh_im and hh are required");
  if (!loglike && !rho2_phase_max) return fail(p, SFT_EINVAL, "at least one of loglike, rho2_phase_max must be non-NULL");
  CU(p, cudaSetDevice(p->d.device));
  const size_t b = (size_t)nT * sizeof(double);
  const double *d_xh = xh, *d_xi = xh_im, *d_hh = hh;
  double *d_l = loglike, *d_r = rho2_phase_max;
  if (mem == SFT_MEM_HOST) {
    sft_status st = grow(p, &p->d_out, &p->out_bytes, 5 * b);
    if (st != SFT_OK) return st;
    double *q = (double *)p->d_out;
    CU(p, cudaMemcpyAsync(q, xh, b, cudaMemcpyHostToDevice, p->stream));
    CU(p, cudaMemcpyAsync(q + nT, xh_im, b, cudaMemcpyHostToDevice, p->stream));
    CU(p, cudaMemcpyAsync(q + 2 * nT, hh, b, cudaMemcpyHostToDevice, p->stream));
    d_xh = q; d_xi = q + nT; d_hh = q + 2 * nT;
    d_l = loglike ? q + 3 * nT : nullptr;
    d_r = rho2_phase_max ? q + 4 * nT : nullptr;
  }
  sftk::sft_statistics_kernel<<<(unsigned)((nT + 255) / 256), 256, 0, p->stream>>>(nT, d_xh, d_xi, d_hh, d_l, d_r);
  p->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "statistics kernel launch: %s", cudaGetErrorString(e));
  if (mem == SFT_MEM_HOST) {
    CU(p, cudaStreamSynchronize(p->stream));
    if (loglike) CU(p, cudaMemcpyAsync(loglike, d_l, b, cudaMemcpyDeviceToHost, p->stream));
    if (rho2_phase_max) CU(p, cudaMemcpyAsync(rho2_phase_max, d_r, b, cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
  }
  return SFT_OK;
}

// Validity flags of Eq.(33)-(34) P:244-248 per template (no data needed).
SFT_API sft_status sft_validity(sft_plan *p, int64_t nT, const double *params, double delta_max, double *delta_eff,
                                uint8_t *flags, int32_t mem) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (nT < 0) return fail(p, SFT_EINVAL, "n_templates < 0");
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(p, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  if (nT == 0) return SFT_OK;
  if (!params) return fail(p, SFT_EINVAL, "params is required");
  if (!delta_eff && !flags) return fail(p, SFT_EINVAL, "at least one of delta_eff, flags must be non-NULL");
  if (!(delta_max >= 0.0)) return fail(p, SFT_EINVAL, "delta_max must be >= 0");
  if (nT > (1ll << 31) - 1) return fail(p, SFT_EINVAL, "n_templates too large");
  CU(p, cudaSetDevice(p->d.device));
  KParams k;
  fill_kparams(p, k);
  k.nT = nT;
  double *d_de = delta_eff;
  unsigned char *d_fl = flags;
  const size_t b_de = (size_t)nT * sizeof(double), b_par = (size_t)nT * SFT_NPARAM * sizeof(double);
  sft_status st;
  if (mem == SFT_MEM_HOST) {
    st = grow(p, (void **)&p->d_params, &p->params_bytes, b_par);
    if (st != SFT_OK) return st;
    st = grow(p, &p->d_out, &p->out_bytes, b_de + (size_t)nT + 256);
    if (st != SFT_OK) return st;
    CU(p, cudaMemcpyAsync(p->d_params, params, b_par, cudaMemcpyHostToDevice, p->stream));
    k.params = p->d_params;
    d_de = (double *)p->d_out;
    d_fl = (unsigned char *)p->d_out + b_de;
  } else {
    k.params = params;
  }
  sftk::sft_validity_kernel<<<(unsigned)((nT + 127) / 128), 128, 0, p->stream>>>(k, delta_max, d_de, d_fl);
  p->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "validity kernel launch: %s", cudaGetErrorString(e));
  if (mem == SFT_MEM_HOST) {
    st = grow_pinned(p, b_de + (size_t)nT);
    if (st != SFT_OK) return st;
    CU(p, cudaMemcpyAsync(p->h_pin, d_de, b_de + (size_t)nT, cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    if (delta_eff) memcpy(delta_eff, p->h_pin, b_de);
    if (flags) memcpy(flags, (char *)p->h_pin + b_de, (size_t)nT);
  }
  return SFT_OK;
}

// F-statistic, Eq.(10)-(13) P:107-122: one pass of the fused kernel (MODE 2) accumulates the seven sums per template.
SFT_API sft_status sft_fstat(sft_plan *p, int64_t nT, const double *params, double *twoF, double *xnu, double *mnu, int32_t mem) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (nT < 0) return fail(p, SFT_EINVAL, "n_templates < 0");
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(p, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  if (nT == 0) return SFT_OK;
  if (!params || !twoF) return fail(p, SFT_EINVAL, "params and twoF are required");
  if (p->d.response != SFT_RESP_TABLE)
    return fail(p, SFT_EINVAL, "sft_fstat needs a plan with SFT_RESP_TABLE: the table holds the antenna-pattern functions (a, b)");
  if (p->d.n_channels > 2) return fail(p, SFT_EUNSUPPORTED, "sft_fstat: at most 2 channels in this build");
  KParams k;
  sft_status st = prepare(p, nT, params, mem, k, false, 7);
  if (st != SFT_OK) return st;
  const size_t b_vec = (size_t)nT * sizeof(double);
  // scratch: the 7 reduced sums, then (host calls) the 1 + 4 + 3 output vectors
  st = grow(p, &p->d_out, &p->out_bytes, 15 * b_vec + 256);
  if (st != SFT_OK) return st;
  double *sums = (double *)p->d_out, *d_F = twoF, *d_x = xnu, *d_m = mnu;
  if (mem == SFT_MEM_HOST) {
    d_F = sums + 7 * nT;
    d_x = xnu ? d_F + nT : nullptr;
    d_m = mnu ? d_F + 5 * nT : nullptr;
  }
  k.kc_out = nullptr;
  k.path_counts = nullptr;
  cudaError_t e = launch_main(p, k, 2);
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "main kernel launch: %s", cudaGetErrorString(e));
  sftk::RedOut ro;
  for (int i = 0; i < 7; ++i) ro.q[i] = sums + (size_t)i * nT;
  sftk::sft_reduce_kernel<<<dim3((unsigned)((nT + 31) / 32), 7), 32 * sftk::RED_SLICES, 0, p->stream>>>(p->part, nT, k.n_chunks, 7, ro);
  sftk::sft_fstat_kernel<<<(unsigned)((nT + 255) / 256), 256, 0, p->stream>>>(nT, sums, d_F, d_x, d_m);
  p->launches += 2;
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "reduce / F-statistic kernel launch: %s", cudaGetErrorString(e));
  if (mem == SFT_MEM_HOST) {
    st = grow_pinned(p, 8 * b_vec);
    if (st != SFT_OK) return st;
    double *h = (double *)p->h_pin;
    CU(p, cudaMemcpyAsync(h, d_F, 8 * b_vec, cudaMemcpyDeviceToHost, p->stream));
    CU(p, cudaStreamSynchronize(p->stream));
    memcpy(twoF, h, b_vec);
    if (xnu) memcpy(xnu, h + nT, 4 * b_vec);
    if (mnu) memcpy(mnu, h + 5 * nT, 3 * b_vec);
  }
  return SFT_OK;
}

SFT_API sft_status sft_cumulative_snr(sft_plan *p, int64_t nT, const double *params, float *snr, float *cum_xh,
                                         float *cum_hh, int32_t mem) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (nT < 0) return fail(p, SFT_EINVAL, "n_templates < 0");
  if (mem != SFT_MEM_HOST && mem != SFT_MEM_DEVICE) return fail(p, SFT_EINVAL, "mem must be SFT_MEM_HOST or SFT_MEM_DEVICE");
  if (nT == 0) return SFT_OK;
  if (!params) return fail(p, SFT_EINVAL, "params is required");
  if (!snr && !cum_xh && !cum_hh) return fail(p, SFT_EINVAL, "at least one of snr, cum_xh, cum_hh must be non-NULL");
  const size_t N = p->d.n_sft, mat = (size_t)nT * N * sizeof(float);
  const int n_out = (snr != nullptr) + (cum_xh != nullptr) + (cum_hh != nullptr);
  sft_status st = SFT_OK;
  if (mem == SFT_MEM_DEVICE) {
    KParams k;
    st = prepare(p, nT, params, mem, k, true);
    if (st != SFT_OK) return st;
    k.out_snr = snr;
    k.out_cx = cum_xh;
    k.out_ch = cum_hh;
#ifdef SFT_CHECKED
    k.n_out = (unsigned long long)nT * N;
#endif
    cudaError_t e = launch_main(p, k, 1);
    if (e != cudaSuccess) return fail(p, SFT_ECUDA, "main kernel launch: %s", cudaGetErrorString(e));
    return SFT_OK;
  }
  // Host outputs: the bank is cut into slabs of templates; slab i + 1 is computed while the matrices of slab i travel to the
  // host on a second stream (the output, 4 n_sft bytes per template and matrix, is what bounds this call end to end).
  // One slab when the whole output is small.
  long long slab = p->slab_user;
  if (slab <= 0) slab = (long long)((64u << 20) / (N * sizeof(float)));            // ~64 MB per matrix and slab
  slab = (slab / 32) * 32;
  if (slab < 32) slab = 32;
  if (slab > nT) slab = nT;
  if (slab < nT && !p->copy_stream) {
    CU(p, cudaSetDevice(p->d.device));
    CU(p, cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) CU(p, cudaEventCreateWithFlags(&p->ev_slab[i], cudaEventDisableTiming));
  }
  st = grow(p, &p->d_out, &p->out_bytes, (size_t)n_out * mat);
  if (st != SFT_OK) return st;
  float *q = (float *)p->d_out;
  float *d_snr = snr ? q : nullptr; if (snr) q += (size_t)nT * N;
  float *d_cx = cum_xh ? q : nullptr; if (cum_xh) q += (size_t)nT * N;
  float *d_ch = cum_hh ? q : nullptr;
  float *const dev[3] = {d_snr, d_cx, d_ch};
  float *const host[3] = {snr, cum_xh, cum_hh};
  auto copy_slab = [&](long long t0, long long n, int i) -> cudaError_t {          // slab i: after its kernel (ev_slab[i & 1])
    cudaStream_t cs = slab < nT ? p->copy_stream : p->stream;
    cudaError_t e = cudaSuccess;
    if (slab < nT) e = cudaStreamWaitEvent(cs, p->ev_slab[i & 1], 0);
    for (int j = 0; j < 3 && e == cudaSuccess; ++j)
      if (host[j]) e = cudaMemcpyAsync(host[j] + (size_t)t0 * N, dev[j] + (size_t)t0 * N, (size_t)n * N * sizeof(float), cudaMemcpyDeviceToHost, cs);
    return e;
  };
  long long prev_t0 = 0, prev_n = 0;
  int i = 0;
  for (long long t0 = 0; t0 < nT; t0 += slab, ++i) {
    const long long n = nT - t0 < slab ? nT - t0 : slab;
    KParams k;
    st = prepare(p, n, params + (size_t)t0 * SFT_NPARAM, mem, k, true);
    if (st != SFT_OK) break;
    k.out_snr = d_snr ? d_snr + (size_t)t0 * N : nullptr;
    k.out_cx = d_cx ? d_cx + (size_t)t0 * N : nullptr;
    k.out_ch = d_ch ? d_ch + (size_t)t0 * N : nullptr;
#ifdef SFT_CHECKED
    k.n_out = (unsigned long long)n * N;
#endif
    cudaError_t e = launch_main(p, k, 1);
    if (e == cudaSuccess && slab < nT) e = cudaEventRecord(p->ev_slab[i & 1], p->stream);
    // the previous slab's copy is issued after this slab's kernel: with pageable host memory cudaMemcpyAsync blocks the host
    if (e == cudaSuccess && i > 0) e = copy_slab(prev_t0, prev_n, i - 1);
    if (e != cudaSuccess) { st = fail(p, SFT_ECUDA, "cumulative slab %d: %s", i, cudaGetErrorString(e)); break; }
    prev_t0 = t0; prev_n = n;
  }
  if (st == SFT_OK) {
    cudaError_t e = copy_slab(prev_t0, prev_n, i - 1);
    if (e != cudaSuccess) st = fail(p, SFT_ECUDA, "cumulative slab %d copy: %s", i - 1, cudaGetErrorString(e));
  }
  // (on an error part of the slabs may already have been written to the host matrices)
  cudaError_t e1 = p->copy_stream ? cudaStreamSynchronize(p->copy_stream) : cudaSuccess;
  cudaError_t e2 = cudaStreamSynchronize(p->stream);
  if (st == SFT_OK && (e1 != cudaSuccess || e2 != cudaSuccess))
    st = fail(p, SFT_ECUDA, "cumulative: %s", cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
  return st;
}

// ---------------------------------------------------------------------------------------------
SFT_API sft_status sft_measure_alu_peaks(int32_t device, double *out, int32_t n_out) {
  g_create_err[0] = 0;
  if (!out || n_out < 1) return fail(nullptr, SFT_EINVAL, "sft_measure_alu_peaks: out is NULL or n_out < 1");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess) return fail(nullptr, SFT_ECUDA, "cudaGetDeviceCount: %s", cudaGetErrorString(e));
  if (device < 0 || device >= ndev) return fail(nullptr, SFT_EINVAL, "device %d not in 0..%d", device, ndev - 1);
  CU(nullptr, cudaSetDevice(device));
  cudaDeviceProp prop;
  CU(nullptr, cudaGetDeviceProperties(&prop, device));
  float *d = nullptr;
  CU(nullptr, cudaMalloc((void **)&d, 64));
  cudaEvent_t e0, e1;
  CU(nullptr, cudaEventCreate(&e0));
  CU(nullptr, cudaEventCreate(&e1));
  const int blocks = prop.multiProcessorCount * 8, threads = 256;
  const double lane_ops = (double)blocks * threads * sftk::PEAK_ITERS * sftk::PEAK_ILP;
  double res[5] = {0, 0, 0, 0, 0};
  for (int which = 0; which < 5; ++which) {
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
      cudaEventRecord(e0, 0);
      switch (which) {
        case 0: sftk::peak_ffma_kernel<<<blocks, threads>>>(d, 1.0000001f, 1e-9f); break;
        case 1: sftk::peak_ffma2_kernel<<<blocks, threads>>>(d, 1.0000001f, 1e-9f); break;
        case 2: sftk::peak_dfma_kernel<<<blocks, threads>>>(d, 1.0000001, 1e-9); break;
        case 3: sftk::peak_mufu_kernel<<<blocks, threads>>>(d, 1.5f); break;
        default: sftk::peak_mix_kernel<<<blocks, threads>>>(d, 1.0000001f, 1e-9f); break;
      }
      cudaEventRecord(e1, 0);
      cudaError_t es = cudaEventSynchronize(e1);
      if (es != cudaSuccess) { cudaFree(d); return fail(nullptr, SFT_ECUDA, "peak kernel: %s", cudaGetErrorString(es)); }
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      if (rep > 0 && ms < best) best = ms;
    }
    const double mult = which == 1 ? 2.0 : (which == 4 ? 1.25 : 1.0);   // packed: 2 lanes; mix: 8 FFMA + 2 MUFU per 8
    res[which] = lane_ops * mult / (best * 1e-3) / 1e9;
  }
  // out[5]: instructions per clock and scheduler sustained on the moment-table kernel's instruction mix
  double mix_ipc = 0.0;
  {
    const int mblocks = prop.multiProcessorCount * 5;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
      cudaEventRecord(e0, 0);
      sftk::peak_mix_table_kernel<<<mblocks, 128>>>(d, 1.0000001f, 1e-9f);
      cudaEventRecord(e1, 0);
      if (cudaEventSynchronize(e1) != cudaSuccess) break;
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      if (rep > 0 && ms < best) best = ms;
    }
    const double warp_instr = (double)mblocks * 4 * sftk::MIXT_ITERS * sftk::MIXT_INSTR;
    const double sched_clocks = best * 1e-3 * (double)prop.clockRate * 1e3 * prop.multiProcessorCount * 4;
    mix_ipc = warp_instr / sched_clocks;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  for (int i = 0; i < n_out && i < 5; ++i) out[i] = res[i];
  if (n_out > 5) out[5] = mix_ipc;
  return SFT_OK;
}

// ---------------------------------------------------------------------------------------------
// sft_inner_products_static: sft_inner_products for callers that may not allocate (CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc).  The scratch of the call - per-template constants td/tf, the chunk totals `part` that
// sft_reduce_kernel sums, the work-unit counter - lives in the file-scope device array below instead of the plan's grown
// buffers; every GPU that loads the library holds SFT_STATIC_SCRATCH_BYTES of it until exit.
//   In host code `g_static_scratch` is the host-side stand-in of the symbol, NOT a device address: the address on a device
// comes from cudaGetSymbolAddress with that device current (static_scratch_ptr, once per device).
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_static_scratch[SFT_STATIC_SCRATCH_BYTES];

namespace {
constexpr int STATIC_MAX_DEV = 64;
constexpr size_t STATIC_HEAD = 256;                       // [0, 256): work-unit counter (zeroed by sft_tmpl_kernel on every call)
std::mutex g_static_mu;
unsigned char *g_static_ptr[STATIC_MAX_DEV] = {nullptr};

constexpr size_t align256(size_t b) { return (b + 255) & ~size_t(255); }

// device address of g_static_scratch on `device` (made current here); resolved once per device
cudaError_t static_scratch_ptr(int device, unsigned char **out) {
  if (device < 0 || device >= STATIC_MAX_DEV) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mu);
  cudaError_t e = cudaSetDevice(device);
  if (e != cudaSuccess) return e;
  if (!g_static_ptr[device]) {
    void *q = nullptr;
    e = cudaGetSymbolAddress(&q, g_static_scratch);
    if (e != cudaSuccess) return e;
    g_static_ptr[device] = (unsigned char *)q;
  }
  *out = g_static_ptr[device];
  return cudaSuccess;
}
}  // namespace

SFT_API sft_status sft_static_setup(int32_t device, int64_t *scratch_bytes) {
  g_create_err[0] = 0;
  unsigned char *q = nullptr;
  const cudaError_t e = static_scratch_ptr(device, &q);
  if (e != cudaSuccess) return fail(nullptr, e == cudaErrorInvalidDevice ? SFT_EINVAL : SFT_ECUDA, "static scratch of device %d: %s", device, cudaGetErrorString(e));
  if (scratch_bytes) *scratch_bytes = (int64_t)SFT_STATIC_SCRATCH_BYTES;
  return SFT_OK;
}

SFT_API sft_status sft_inner_products_static(sft_plan *p, int64_t nT, const double *params, double *xh, double *hh, double *xh_im) {
  if (!p) return SFT_EINVAL;
  p->err[0] = 0;
  if (nT < 0) return fail(p, SFT_EINVAL, "n_templates < 0");
  if (nT == 0) return SFT_OK;
  if (!params || !xh || !hh) return fail(p, SFT_EINVAL, "params, xh and hh are required (device pointers)");
  if (nT > SFT_STATIC_MAX_TEMPLATES)
    return fail(p, SFT_EUNSUPPORTED, "sft_inner_products_static: n_templates = %lld exceeds SFT_STATIC_MAX_TEMPLATES = %d "
                "(static scratch of %d bytes); split the bank or use sft_inner_products", (long long)nT,
                (int)SFT_STATIC_MAX_TEMPLATES, (int)SFT_STATIC_SCRATCH_BYTES);
  for (int c = 0; c < p->d.n_channels; ++c)
    if (!p->loaded[c]) return fail(p, SFT_ENODATA, "channel %d has no data (call sft_load_data)", c);
  unsigned char *base = nullptr;
  cudaError_t e = static_scratch_ptr(p->d.device, &base);          // (makes the plan's device current)
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "static scratch of device %d: %s", p->d.device, cudaGetErrorString(e));
  // carve the scratch: counter | td [TD_N][nT] fp64 | tf [TF_N][nT] fp32 | part [n_chunks][3][nT] fp64
  const size_t o_td = STATIC_HEAD, o_tf = o_td + align256((size_t)sftk::TD_N * nT * sizeof(double));
  const size_t o_part = o_tf + align256((size_t)sftk::TF_N * nT * sizeof(float));
  const size_t row = 3 * (size_t)nT * sizeof(double);                // chunk totals of one chunk
  if (o_part + row > (size_t)SFT_STATIC_SCRATCH_BYTES) return fail(p, SFT_EUNSUPPORTED, "static scratch too small for %lld templates", (long long)nT);
  const long long max_chunks = (long long)(((size_t)SFT_STATIC_SCRATCH_BYTES - o_part) / row);
  KParams k;
  fill_kparams(p, k);
  k.nT = nT;
  k.n_tgroups = (int)((nT + 31) / 32);
  // SFTs per work unit: the rule of prepare(), with the number of chunks capped by what the scratch holds
  const long long target_units = 16ll * p->n_sm * 24;
  long long want_chunks = (target_units + k.n_tgroups - 1) / k.n_tgroups;
  if (want_chunks > max_chunks) want_chunks = max_chunks;
  if (want_chunks < 1) want_chunks = 1;
  int chunk = (int)((k.n_sft + want_chunks - 1) / want_chunks);
  if (chunk < 32) chunk = 32;
  chunk = ((chunk + 31) / 32) * 32;                                  // aligned to the blocks of 32 SFT slots (fast path, table layout)
  if (chunk > k.n_sft) chunk = k.n_sft;
  k.chunk = chunk;
  k.n_chunks = (k.n_sft + chunk - 1) / chunk;
  if (k.n_chunks > max_chunks) return fail(p, SFT_EUNSUPPORTED, "static scratch too small: %d chunks of %d SFTs needed, room for %lld", k.n_chunks, chunk, max_chunks);
  k.n_items = k.n_tgroups * k.n_chunks;
  k.counter = (int *)base;
  double *td = (double *)(base + o_td);
  float *tf = (float *)(base + o_tf);
  double *part = (double *)(base + o_part);
  k.td = td;
  k.tf = tf;
  k.part = part;
  k.params = params;
#ifdef SFT_CHECKED
  k.n_part = (unsigned long long)k.n_chunks * 3 * nT;
#endif
  // nothing in the scratch needs to start at zero except the counter, which sft_tmpl_kernel clears; td, tf and every
  // (chunk, quantity, template) entry of part that the reduction reads are written by this call before they are read
  sftk::sft_tmpl_kernel<<<(unsigned)((nT + 127) / 128), 128, 0, p->stream>>>(k, td, tf);
  p->launches++;
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "template kernel launch: %s", cudaGetErrorString(e));
  e = launch_main(p, k, 0);
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "main kernel launch: %s", cudaGetErrorString(e));
  sftk::RedOut ro = {{xh, hh, xh_im, nullptr, nullptr, nullptr, nullptr}};
  sftk::sft_reduce_kernel<<<dim3((unsigned)((nT + 31) / 32), 3), 32 * sftk::RED_SLICES, 0, p->stream>>>(part, nT, k.n_chunks, 3, ro);
  p->launches++;
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, SFT_ECUDA, "reduce kernel launch: %s", cudaGetErrorString(e));
  return SFT_OK;
}
