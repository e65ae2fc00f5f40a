// sft_table.cuh - the moment-table evaluator of libsft_b200.so: load-time kernels (sm_100a).
//
// Idea ("moment tables").  For one (channel, SFT) the contraction of rows A4+A6,
//
//   S1(xp, b) = sum_{m=-K..K} D_{kc+m} J_m(xp, b),
//   J_m(xp, b) = (-1)^m int_{-1/2}^{1/2} exp(i (2 pi (xp - m) v + pi b v^2)) dv        (Eq.(28) P:215 about the SFT mid-point)
//
// is a smooth (entire) function of the template's fractional bin offset xp = f_a T + b/2 - k_c and of
// b = fdot T^2: with E(v) = sum_m D_{kc+m} (-1)^m e^{-2 pi i m v} it is int e^{i(2 pi xp v + pi b v^2)} E(v) dv.
// Expanding about a node xj (xp = xj + delta) and b = 0,
//
//   S1 = sum_{p,n} (i a)^p/p! (i beta)^n/n! M_{p+2n}(kc, xj),   a = 2 pi delta, beta = pi b,
//   M_q(kc, xj) = sum_m D_{kc+m} (-1)^m rho_q(xj - m),   rho_q(a') = int_{-1/2}^{1/2} v^q e^{2 pi i a' v} dv,
//
// with |v| <= 1/2 the terms fall like (pi delta)^p/p! (pi b/4)^n/n!.  The moments M_q do not depend on
// the template: they are computed ONCE per data set (as the SFTs themselves are) for
// every window position kc and TAB_R nodes per bin, q = 0..TAB_Q, and kept in HBM; a template then
// needs 64 bytes and ~20 packed FMAs per (SFT, channel) instead of evaluating 2K+1 kernel coefficients.
// Truncation error at TAB_R = 4 (measured against fp64 quadrature, moments stored as complex64), relative to
// sqrt(sum |D|^2):  tier 1, q <= 7:  4e-7 at |b| = 0.12 (3e-8 at 0.056);  tier 2, q <= 15:  2e-8 up to |b| = 0.5,
// 2.4e-7 at |b| = 1.0 (7e-6 at 1.5).  |b| > B_TABLE2 = 1 takes the direct evaluator of sft_kernels.cuh.
//
// The <h,h> sum H(kc, xp, b) = sum_m u_{kc+m} |J_m|^2 (u = S_ref/S_k) does not depend on the data at
// all; it is even in b and tabulated per window position on HTAB_R = 64 nodes per bin as
//   H = sum_{P<=3} a^P sum_N beta^(2N) h_{P,2N}:  N <= 1: relative error < 3e-7 for |b| <= 0.12;  N <= 3: 9e-8 at |b| = 1
// (|a| <= 2 pi / 128 = 0.05 about a node: the cubic in a is exact to ~1e-8; 32 bytes and 7 FMAs per (template, SFT) in tier 1).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sftk {

constexpr int TAB_R = 4;      // nodes per bin of the data-moment table
constexpr int TAB_Q = 15;     // highest moment kept (TAB_Q + 1 complex64 = 128 bytes per node)
constexpr int TAB_Q1 = 7;     // highest moment used by tier 1 (the first 64 bytes of a node)
constexpr int HTAB_R = 64;    // nodes per bin of the <h,h> table
constexpr int HTAB_SHIFT = 4; // HTAB_R = TAB_R << HTAB_SHIFT: the data-moment node of an <h,h> node is cellH >> HTAB_SHIFT
constexpr int HTAB_P = 3;     // highest power of a kept (|a| <= 2 pi / 128: the a^4 term is below 1e-7 of H)
constexpr int HTAB_NB = 4;    // powers of beta^2 kept: beta^0, beta^2, beta^4, beta^6 (tier 1 uses the first two)
constexpr int HTAB_W = 16;    // floats per node: h_{0..3,0}, h_{0..3,2}, h_{0..3,4}, h_{0..3,6} (tier 1 reads the first 32 bytes)
static_assert(HTAB_R == (TAB_R << HTAB_SHIFT) && HTAB_W == HTAB_NB * (HTAB_P + 1) && HTAB_W % 4 == 0, "table geometry");
// Tier 1 reads a compact <h,h> node instead: 16 bytes {h_00, h_10, h_20, h_02} on HT1_R = 256 nodes per bin,
//   H = h_00 + a (h_10 + a h_20) + beta^2 h_02,   |a| <= 2 pi / 512:
// the cubic in a is below 4e-9 of H and the beta^2 term (|h_02| <~ 3e-5: the power only moves between neighbouring bins) may be
// taken at the node; measured against fp64 quadrature with flat and steep PSDs: 2.4e-8 relative for |b| <= 0.12.
constexpr int HT1_R = 256;    // nodes per bin of the compact tier-1 <h,h> table
constexpr int HT1_SHIFT = 6;  // HT1_R = TAB_R << HT1_SHIFT
static_assert(HT1_R == (TAB_R << HT1_SHIFT), "table geometry");
constexpr float B_TABLE = 0.12f;    // tier 1: moments q <= 7, H to beta^2
constexpr float B_TABLE2 = 1.0f;    // tier 2: moments q <= 15, H to beta^6

#ifndef SFT_MAIN_ONLY
// sigma_q(a') with rho_q = sigma_q (q even), i sigma_q (q odd):  sigma_q = int v^q cos(w v) dv (q even), int v^q sin(w v) dv (q odd),
// w = 2 pi a', over [-1/2, 1/2].  |a'| >= 1.5: integration by parts upwards in q (each step multiplies
// the error by q/w < 1); below: power series in w (|w|/2 < 4.8: 40 terms leave < 1e-17).
template <int NQ>
__device__ void sigma_moments(double ap, double (&sig)[NQ]) {
  const double w = 6.283185307179586 * ap;
  if (fabs(ap) >= 1.5) {
    double s, c;
    sincospi(ap, &s, &c);              // sin(w/2), cos(w/2)
    const double iw = 1.0 / w;
    double hq = 1.0;                   // (1/2)^q
    sig[0] = 2.0 * s * iw;
#pragma unroll
    for (int q = 1; q < NQ; ++q) {
      hq *= 0.5;
      sig[q] = (q & 1) ? (-2.0 * hq * c + q * sig[q - 1]) * iw : (2.0 * hq * s - q * sig[q - 1]) * iw;
    }
  } else {
#pragma unroll
    for (int q = 0; q < NQ; ++q) sig[q] = 0.0;
    double term = 1.0;                 // w^k / k!
    for (int k = 0; k < 44; ++k) {
      const double sgn = ((k >> 1) & 1) ? -1.0 : 1.0;        // (-1)^floor(k/2)
      double hp = ldexp(1.0, -(k + 1));                      // (1/2)^(q+k+1), q = 0
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        if (((q + k) & 1) == 0) sig[q] += sgn * term * 2.0 * hp / (double)(q + k + 1);
        hp *= 0.5;
      }
      term *= w / (double)(k + 1);
    }
  }
}

// P-table: ptab[mi][cell][q] = (-1)^m rho_q(xj_cell - m) as complex64, m = mi - K.
__global__ void sft_ptab_kernel(int K, float2 *ptab) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (2 * K + 1) * TAB_R) return;
  const int mi = idx / TAB_R, cell = idx - mi * TAB_R, m = mi - K;
  const double xj = ((double)cell + 0.5) / TAB_R - 0.5;
  double sig[TAB_Q + 1];
  sigma_moments<TAB_Q + 1>(xj - (double)m, sig);
  const double sg = (m & 1) ? -1.0 : 1.0;
#pragma unroll
  for (int q = 0; q <= TAB_Q; ++q) {
    const double v = sg * sig[q];
    ptab[(size_t)idx * (TAB_Q + 1) + q] = (q & 1) ? make_float2(0.f, (float)v) : make_float2((float)v, 0.f);
  }
}

// Data-moment table of one channel.  Layout per block of 32 SFT slots, tblk[a >> 5] = {float4 index of the block's first row,
// kb, W, float4 per row}: the row of SFT a holds the nodes of the W window positions kb .. kb + W - 1 (counted from k_lo - K),
// node = (kcidx - kb) * TAB_R + cell, TAB_Q + 1 complex64 moments each.  Grid: n_rows * bpr blocks (bpr = blocks per row for
// the widest block); `a_first` = SFT slot of the first row handled (sft_append_sfts builds a range), Dp0 = its padded whitened
// row in copy 0 of the pair-planar store (neighbouring threads share a window: L1 broadcast), ptab through L1.
__global__ void __launch_bounds__(256) sft_mtab_kernel(const float4 *Dp0, int npair, const int4 *tblk, int a_first, int K,
                                                       const float2 *ptab, unsigned bpr, float2 *mtab) {
  const unsigned al = blockIdx.x / bpr, bx = blockIdx.x - al * bpr;
  const int a = a_first + (int)al;
  const int4 tb = __ldg(tblk + (a >> 5));
  const float4 *src = Dp0 + (size_t)al * npair;
  constexpr int nq = TAB_Q + 1, per_bin = TAB_R * nq;
  const int o = bx * blockDim.x + threadIdx.x;                // (node, q) flattened
  if (o >= tb.z * per_bin) return;
  const int kcl = o / per_bin, cq = o - kcl * per_bin;         // cq = cell * nq + q
  const float2 *pp = ptab + cq;
  float re = 0.f, im = 0.f;
  const int nb = 2 * K + 1;
  for (int mi = 0; mi < nb; ++mi) {
    const int j = tb.y + kcl + 2 + mi;                         // window start j0 = kcidx + 2
    const float4 d4 = __ldg(src + (j >> 1));
    const float dx = (j & 1) ? d4.y : d4.x, dy = (j & 1) ? d4.w : d4.z;
    const float2 pv = __ldg(pp + (size_t)mi * per_bin);
    re = fmaf(dx, pv.x, re); re = fmaf(-dy, pv.y, re);
    im = fmaf(dx, pv.y, im); im = fmaf(dy, pv.x, im);
  }
  mtab[2 * ((size_t)(unsigned)tb.x + (size_t)(a & 31) * (unsigned)tb.w) + o] = make_float2(re, im);
}

// <h,h> table of one channel: htab[nodeH][HTAB_W], nodeH = kcidx * HTAB_R + cell.  One block per node,
// threads over the 2K+1 bins; fp64.  rho_q = sigma_q (q even), i sigma_q (q odd), and p + 2n has the parity of
// p, so the coefficient of a^p beta^n in J_m is  c_{p,n} = (-1)^m e_p i^n sigma_{p+2n} / (p! n!)  with the real
// sign e_p = i^p (p odd ? i : 1) = (-1)^ceil(p/2); the polynomial of |J_m|^2 has the coefficients
//   h_{P,2N} = sum_{p+p'=P} sum_{n+n'=2N} e_p e_p' (-1)^((n-n')/2) sigma_{p+2n} sigma_{p'+2n'} / (p! p'! n! n'!)
// (odd powers of beta cancel: |J|^2 is even in b).
__global__ void __launch_bounds__(64) sft_htab_kernel(const float2 *ub0, int K, float *htab) {
  constexpr int NMAX = 2 * (HTAB_NB - 1);         // highest single power of beta: 6
  constexpr int NQ = HTAB_P + 2 * NMAX + 1;       // sigma_0 .. sigma_{P + 2 NMAX}
  constexpr int NH = HTAB_NB * (HTAB_P + 1);
  __shared__ double red[NH];
  const int node = blockIdx.x, kcidx = node / HTAB_R, cell = node - kcidx * HTAB_R;
  if (threadIdx.x < NH) red[threadIdx.x] = 0.0;
  __syncthreads();
  const double xj = ((double)cell + 0.5) / HTAB_R - 0.5;
  const double fact[7] = {1.0, 1.0, 2.0, 6.0, 24.0, 120.0, 720.0};
  for (int mi = threadIdx.x; mi <= 2 * K; mi += blockDim.x) {
    const int j = kcidx + 2 + mi;
    const float2 u2 = __ldg(ub0 + (j >> 1));
    const double u = (j & 1) ? (double)u2.y : (double)u2.x;
    if (u == 0.0) continue;
    double sig[NQ];
    sigma_moments<NQ>(xj - (double)(mi - K), sig);
    for (int P = 0; P <= HTAB_P; ++P) {
      for (int N2 = 0; N2 < HTAB_NB; ++N2) {
        double acc = 0.0;
        for (int p = 0; p <= P; ++p) {
          const int pp = P - p;
          const double sgn_p = ((((p + 1) >> 1) + ((pp + 1) >> 1)) & 1) ? -1.0 : 1.0;      // e_p e_p'
          for (int n = 0; n <= 2 * N2; ++n) {
            const int nn = 2 * N2 - n;
            if (n > NMAX || nn > NMAX) continue;
            const int hd = n - nn;                                                        // even
            const double sgn_n = ((hd / 2) & 1) ? -1.0 : 1.0;                             // (-1)^((n-n')/2)
            acc += sgn_p * sgn_n * sig[p + 2 * n] * sig[pp + 2 * nn] / (fact[p] * fact[pp] * fact[n] * fact[nn]);
          }
        }
        atomicAdd(&red[N2 * (HTAB_P + 1) + P], u * acc);
      }
    }
  }
  __syncthreads();
  if (threadIdx.x < HTAB_W) htab[(size_t)node * HTAB_W + threadIdx.x] = threadIdx.x < NH ? (float)red[threadIdx.x] : 0.f;
}

// Compact tier-1 <h,h> table of one channel: htab1[nodeH] = {h_00, h_10, h_20, h_02}, nodeH = kcidx * HT1_R + cell (the
// coefficients of sft_htab_kernel's expansion that tier 1 keeps):
//   h_00 = sum u s0^2,  h_10 = -2 sum u s0 s1,  h_20 = sum u (s1^2 - s0 s2),  h_02 = sum u (s2^2 - s0 s4),   s_q = sigma_q(xj - m).
__global__ void __launch_bounds__(64) sft_htab1_kernel(const float2 *ub0, int K, float4 *htab1) {
  __shared__ double red[4];
  const int node = blockIdx.x, kcidx = node / HT1_R, cell = node - kcidx * HT1_R;
  if (threadIdx.x < 4) red[threadIdx.x] = 0.0;
  __syncthreads();
  const double xj = ((double)cell + 0.5) / HT1_R - 0.5;
  for (int mi = threadIdx.x; mi <= 2 * K; mi += blockDim.x) {
    const int j = kcidx + 2 + mi;
    const float2 u2 = __ldg(ub0 + (j >> 1));
    const double u = (j & 1) ? (double)u2.y : (double)u2.x;
    if (u == 0.0) continue;
    double sig[5];
    sigma_moments<5>(xj - (double)(mi - K), sig);
    atomicAdd(&red[0], u * sig[0] * sig[0]);
    atomicAdd(&red[1], -2.0 * u * sig[0] * sig[1]);
    atomicAdd(&red[2], u * (sig[1] * sig[1] - sig[0] * sig[2]));
    atomicAdd(&red[3], u * (sig[2] * sig[2] - sig[0] * sig[4]));
  }
  __syncthreads();
  if (threadIdx.x == 0) htab1[node] = make_float4((float)red[0], (float)red[1], (float)red[2], (float)red[3]);
}

#endif  // SFT_MAIN_ONLY

}  // namespace sftk
