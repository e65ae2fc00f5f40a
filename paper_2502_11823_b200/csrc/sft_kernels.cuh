// sft_kernels.cuh - device code of libsft_b200.so (sm_100a).  See include/sft.h for the maths
// and DESIGN.md for the layout; "P:NNN" cites the paper text, "DESIGN xx" a reading in DESIGN.md.
//
// One thread owns one template and walks a chunk of consecutive SFTs; a warp therefore holds 32
// templates at the SAME SFT, so that (i) every data-bin load is a warp-wide broadcast of the same
// few addresses (templates of a bank tile select the same k_c to within a bin), (ii) the branch on
// the chirp parameter b = fdot T^2 (series vs Fresnel form) is warp-uniform, and (iii) the sum over
// SFTs needs no cross-lane traffic at all: it is a private fp64 accumulator per thread.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "fresnel_aux_coeffs.h"

namespace sftk {

constexpr int TILE = 128;            // templates (= threads) per block
constexpr int MAXC = 4;              // SFT_MAX_CHANNELS
constexpr double GMSUN_S = 4.925491025543576e-6;   // G Msun / c^3 [s]
constexpr float PI_F = 3.14159265358979f;

// b = fdot T^2 thresholds of the coefficient evaluator (DESIGN "kernel evaluator"): the power
// series in b about the SFT mid-point truncated after order n has error <= (pi b)^(n+1) /
// ((n+1)! 4^(n+1) (2n+3)); the bounds below keep that under 2e-6.
constexpr float B_ORDER1 = 0.0057f;  // |b| <= : order 1
constexpr float B_ORDER3 = 0.18f;    // |b| <= : order 3; above: closed Fresnel form

struct KParams {
  int C, n_sft, nb, k_lo, kv_lo, kv_hi, K;
  int kernel, pn1, response;
  double T, t0, f_loT, f_hiT, inv_fref;
  double sigma[MAXC];      // sqrt(T / S_ref,c)
  double chi[MAXC];        // SFT_RESP_ANNUAL response phase per channel
  float depth;
  const float2 *D;         // [C][n_sft][nb]   2 conj(x~) sqrt(S_ref) / (sqrt(T) s_a S_k)
  const float *ub2;        // [C][nb]          S_ref / S_k   (0 for invalid bins)
  const float *us2;        // [C][n_sft]       1 / s_a       (0 for gaps)
  const float2 *rtab;      // [C][n_sft]       TABLE: R_{c,a}; ANNUAL: (cos, sin)(2 pi t_a/P + psi_c)
  const double *params;    // [nT][8]
  long long nT;
  int chunk, n_chunks;
  double *part;            // [n_chunks][3][nT] chunk totals (xh, hh, xh_im)
  int *kc_out;             // [nT][C][n_sft] or null
  float *loc_xh, *loc_hh;  // cumulative mode: [nT][n_sft] chunk-local prefix sums
};

__device__ __forceinline__ float rcp_approx(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

template <int N>
__device__ __forceinline__ float horner(const float *c, float s) {
  float r = c[N];
#pragma unroll
  for (int i = N - 1; i >= 0; --i) r = fmaf(r, s, c[i]);
  return r;
}

// Fresnel auxiliary functions g(t), f(t), t >= 0:  C(t) + i S(t) = (1+i)/2 - (g + i f) e^{i pi t^2/2}
// (C, S of Eq.(31)-(32) P:230-236).  Coefficients: gen_fresnel_aux.py.
__device__ __forceinline__ void fresnel_w(float t, float &g, float &f) {
  if (t < 1.0f) {
    const float s = fmaf(2.0f, t, -1.0f);
    f = horner<9>(FA_F0, s);
    g = horner<9>(FA_G0, s);
  } else if (t < 2.0f) {
    const float s = fmaf(2.0f, t, -3.0f);
    f = horner<8>(FA_F1, s);
    g = horner<8>(FA_G1, s);
  } else {
    const float rt = rcp_approx(t);
    const float y = rt * rt;
    const float s = fmaf(8.0f, y, -1.0f);
    const float rp = rt * (1.0f / PI_F);
    f = horner<6>(FA_F2, s) * rp;
    g = horner<6>(FA_G2, s) * rp * y * (1.0f / PI_F);
  }
}

// Per-template constants, fp64 where the phase needs it (the template is "described by 4
// numbers" per SFT; these are the closed-form coefficients of those 4 numbers, DESIGN W1).
struct Tmpl {
  double tc, cTheta, phic_cyc, cphase, cphi, cf, F0T, bscale;
  float cf32, cl, sl;
  float2 AE[MAXC];   // amp (F0/f_ref)^(2/3) sigma_c e^{i(chi_c+beta)}
  bool ok;
};

__device__ __forceinline__ void tmpl_init(const KParams &p, long long t, Tmpl &tm) {
  tm.ok = t < p.nT;
  const double *row = p.params + (tm.ok ? t : 0) * 8;
  const double mc = row[0], eta = row[1], tc = row[2], phic = row[3], amp = row[4];
  const double lam = row[5], beta = row[6];
  const double M = mc * pow(eta, -0.6) * GMSUN_S;             // total mass [s]
  const double inv2pi = 0.15915494309189535;
  tm.tc = tc;
  tm.cTheta = eta / (5.0 * M);
  tm.phic_cyc = phic * inv2pi;
  tm.cphase = (2.0 / eta) * inv2pi;
  tm.cphi = p.pn1 ? (3715.0 / 8064.0 + 55.0 / 96.0 * eta) : 0.0;
  tm.cf = p.pn1 ? (743.0 / 2688.0 + 11.0 / 32.0 * eta) : 0.0;
  const double F0 = 1.0 / (8.0 * 3.141592653589793 * M);
  tm.F0T = F0 * p.T;
  tm.bscale = tm.cTheta * F0 * p.T * p.T;
  tm.cf32 = (float)tm.cf;
  const double A0 = amp * cbrt((F0 * p.inv_fref) * (F0 * p.inv_fref));
  double sl, cl;
  sincos(lam, &sl, &cl);
  tm.cl = (float)cl;
  tm.sl = (float)sl;
#pragma unroll
  for (int c = 0; c < MAXC; ++c) {
    if (c < p.C) {
      double s, co;
      const double ang = (p.response == 2) ? (p.chi[c] + beta) : 0.0;
      sincos(ang, &s, &co);
      const double a = A0 * p.sigma[c];
      tm.AE[c] = make_float2((float)(a * co), (float)(a * s));
    } else {
      tm.AE[c] = make_float2(0.f, 0.f);
    }
  }
}

// The four numbers of P:164 at t_a, reduced for fp32 consumption.
struct Track {
  bool active;
  int kc;        // central bin (DESIGN A5)
  float x;       // f_a T - k_c
  float b;       // fdot_a T^2
  float frac;    // phi_a / 2 pi mod 1, in [-1/2, 1/2]
  float amp;     // (f_a / F0)^(2/3) = Theta^(-1/4) (1 + cf Theta^(-1/4))^(2/3)
};

__device__ __forceinline__ void track_eval(const KParams &p, const Tmpl &tm, int alpha, Track &tr) {
  const double ta = p.t0 + (double)alpha * p.T;
  const double tau = tm.tc - ta;
  tr.active = false;
  tr.kc = -1;
  if (!tm.ok || !(tau > p.T)) return;
  const double theta = tm.cTheta * tau;
  const double q = rsqrt(sqrt(sqrt(theta)));      // Theta^(-1/8)
  const double q2 = q * q, q3 = q2 * q, q4 = q2 * q2, q8 = q4 * q4;
  const double ph = tm.phic_cyc - tm.cphase * (theta * q3) * fma(tm.cphi, q2, 1.0);   // cycles
  const double fT = tm.F0T * q3 * fma(tm.cf, q2, 1.0);
  const double b = tm.bscale * (q8 * q3) * fma(0.625 * tm.cf, q2, 0.375);
  const double y = (p.kernel == 1) ? fma(0.5, b, fT) : fT;   // Fresnel: centre of the swept band
  const double kcd = floor(y + 0.5);
  if (!(fT >= p.f_loT) || !(fT + b <= p.f_hiT)) return;
  tr.active = true;
  tr.kc = (int)kcd;
  tr.x = (float)(fT - kcd);
  tr.b = (float)b;
  tr.frac = (float)(ph - rint(ph));
  const float q2f = (float)q2;
  float a = q2f;
  if (p.pn1) {
    const float e = fmaf(tm.cf32, q2f, 1.0f);
    a *= cbrtf(e * e);
  }
  tr.amp = a;
}

// ---------------------------------------------------------------------------------------------
// Coefficient evaluator + contraction for one (template, SFT): accumulates, per channel,
//   S1 = sum_m D_{k_c+m} I_m     (complex)      S2 = sum_m ub2_{k_c+m} |I_m|^2
// where F(x-m, b) = pref * I_m and `pref` (unit modulus times a real scale) is returned through
// (pr, pi, scale):  F_m = scale * (pr + i pi) * I_m.
//
// Series form (|b| <= B_ORDER3), about the SFT mid-point (DESIGN "kernel evaluator"):
//   F(x-m,b) = e^{i pi (x-m+b/4)} int_{-1/2}^{1/2} e^{i pi (2 a' v + b v^2)} dv,  a' = x + b/2 - m
//            = e^{i pi (x+b/4)} sum_n (i pi b)^n / n! * r_2n(a'),
//   (-1)^m r_j from the forward recurrence of int v^j e^{i w v} dv (w = 2 pi a'), which is stable
//   for |a'| >= 1/2; the central bin (|a'| < 1/2) uses the Taylor series in (pi a')^2.
// b = 0 is the Dirichlet kernel e^{i pi a} sinc(a), Eq.(B2) P:451.
// ---------------------------------------------------------------------------------------------
template <int ORDER>
__device__ __forceinline__ void series_central(float xp, float pb, float &Ir, float &Ii) {
  // r_2n(w) = 4^-n sum_p (-1)^p z^p / ((2p)! (2n+2p+1)),  z = (pi xp)^2 <= (pi/2)^2
  const float z = (PI_F * xp) * (PI_F * xp);
  auto tay = [&](int n) {
    float acc = 0.f;
    float fact[8] = {1.f, 2.f, 24.f, 720.f, 40320.f, 3628800.f, 479001600.f, 87178291200.f};
#pragma unroll
    for (int pp = 7; pp >= 0; --pp) {
      const float c = ((pp & 1) ? -1.f : 1.f) / (fact[pp] * (float)(2 * n + 2 * pp + 1));
      acc = fmaf(acc, z, c);
    }
    return acc;
  };
  const float r0 = tay(0);
  Ir = r0;
  Ii = 0.f;
  if (ORDER >= 1) Ii = pb * (0.25f * tay(1));
  if (ORDER >= 3) {
    Ir = fmaf(-0.5f * pb * pb, 0.0625f * tay(2), Ir);
    Ii = fmaf(-(1.0f / 6.0f) * pb * pb * pb, 0.015625f * tay(3), Ii);
  }
}

template <int ORDER>
__device__ __forceinline__ void series_far(float ap, float S, float C, float pb, float &Ir, float &Ii) {
  const float w = rcp_approx(2.0f * PI_F * ap);   // 1 / omega
  const float r0 = 2.0f * S * w;
  Ir = r0;
  Ii = 0.f;
  if (ORDER >= 1) {
    const float q1 = (r0 - C) * w;
    const float r2 = fmaf(0.5f, S, -2.0f * q1) * w;
    Ii = pb * r2;
    if (ORDER >= 3) {
      const float q3 = fmaf(3.0f, r2, -0.25f * C) * w;
      const float r4 = fmaf(0.125f, S, -4.0f * q3) * w;
      const float q5 = fmaf(5.0f, r4, -0.0625f * C) * w;
      const float r6 = fmaf(0.03125f, S, -6.0f * q5) * w;
      Ir = fmaf(-0.5f * pb * pb, r4, Ir);
      Ii = fmaf(-(1.0f / 6.0f) * pb * pb * pb, r6, Ii);
    }
  }
}

// Closed Fresnel form (Eq.(29)-(30) P:219-226) rewritten with the auxiliary functions so that the
// large phase pi a^2/b cancels analytically (DESIGN "kernel evaluator"):  with l = a sqrt(2/b),
// u = l + sqrt(2b), w(t) = g(t) + i f(t), E = e^{i pi (2x+b)},
//   sqrt(2b) F(a,b) = sgn(l) w(|l|) - E sgn(u) w(|u|) + [l < 0 <= u] (1+i) e^{-i pi a^2/b}.
__device__ __forceinline__ void fresnel_bin(float a, float c1, float c2, float inv_b, float Er, float Ei,
                                            float &Yr, float &Yi) {
  const float l = a * c1;
  const float u = l + c2;
  float gl, fl, gu, fu;
  fresnel_w(fabsf(l), gl, fl);
  fresnel_w(fabsf(u), gu, fu);
  const float sl = (l >= 0.f) ? 1.f : -1.f;
  const float su = (u >= 0.f) ? 1.f : -1.f;
  // E * w(|u|)
  const float er = Er * gu - Ei * fu;
  const float ei = Er * fu + Ei * gu;
  Yr = sl * gl - su * er;
  Yi = sl * fl - su * ei;
  if (l < 0.f && u >= 0.f) {
    float s, c;
    sincospif(a * a * inv_b, &s, &c);     // e^{-i pi a^2/b} = c - i s ;  (1+i)(c - i s) = (c+s) + i(c-s)
    Yr += c + s;
    Yi += c - s;
  }
}

template <int KT, int CT>
__device__ __forceinline__ void pair_contract(const KParams &p, int alpha, const Track &tr,
                                              float (&S1r)[CT], float (&S1i)[CT], float (&S2)[CT],
                                              float &pr, float &pi_, float &scale) {
  const int K = KT > 0 ? KT : p.K;
  const int C = p.C;
#pragma unroll
  for (int c = 0; c < CT; ++c) { S1r[c] = 0.f; S1i[c] = 0.f; S2[c] = 0.f; }
  const bool fres = (p.kernel == 1);
  const float b = fres ? tr.b : 0.f;
  const float x = tr.x;
  const int col0 = tr.kc - p.k_lo;                    // column of the central bin in the store
  const int mlo = max(-K, p.kv_lo - tr.kc), mhi = min(K, p.kv_hi - 1 - tr.kc);
  const float2 *Drow = p.D + (size_t)alpha * p.nb + col0;
  const float *ubrow = p.ub2 + col0;
  const size_t Dstride = (size_t)p.n_sft * p.nb;

  auto accum = [&](int m, float Ir, float Ii) {
    const float mag = fmaf(Ir, Ir, Ii * Ii);
#pragma unroll
    for (int c = 0; c < CT; ++c) {
      if (c < C) {
        const float2 d = __ldg(Drow + c * Dstride + m);
        const float w2 = __ldg(ubrow + c * p.nb + m);
        S1r[c] = fmaf(d.x, Ir, fmaf(-d.y, Ii, S1r[c]));
        S1i[c] = fmaf(d.x, Ii, fmaf(d.y, Ir, S1i[c]));
        S2[c] = fmaf(w2, mag, S2[c]);
      }
    }
  };

  if (fabsf(b) <= B_ORDER3) {
    const float xp = fmaf(0.5f, b, x);
    const float pb = PI_F * b;
    float S, Cc;
    sincospif(xp, &S, &Cc);
    const int ord = (b == 0.f) ? 0 : (fabsf(b) <= B_ORDER1 ? 1 : 3);
    // prefactor e^{i pi (x + b/4)}
    sincospif(fmaf(0.25f, b, x), &pi_, &pr);
    scale = 1.0f;
#pragma unroll
    for (int m = -K; m <= K; ++m) {
      if (m < mlo || m > mhi) continue;
      float Ir, Ii;
      const float ap = xp - (float)m;
      if (fabsf(ap) < 0.5f) {
        if (ord == 0) series_central<0>(ap, pb, Ir, Ii);
        else if (ord == 1) series_central<1>(ap, pb, Ir, Ii);
        else series_central<3>(ap, pb, Ir, Ii);
        // Taylor form carries no (-1)^m; the far form's S, C are those of xp, i.e. include it
        if (m & 1) { Ir = -Ir; Ii = -Ii; }
      } else {
        if (ord == 0) series_far<0>(ap, S, Cc, pb, Ir, Ii);
        else if (ord == 1) series_far<1>(ap, S, Cc, pb, Ir, Ii);
        else series_far<3>(ap, S, Cc, pb, Ir, Ii);
      }
      accum(m, Ir, Ii);
    }
  } else {
    // closed Fresnel form; b < 0: F(a,-|b|) = conj F(-a,|b|)  (DESIGN A10)
    const bool neg = b < 0.f;
    const float ab = fabsf(b);
    const float c1 = sqrtf(2.0f / ab), c2 = sqrtf(2.0f * ab), inv_b = 1.0f / ab;
    const float xs = neg ? -x : x;
    float Er, Ei;
    sincospif(fmaf(2.0f, xs, ab), &Ei, &Er);
    pr = 1.0f;
    pi_ = 0.0f;
    scale = 1.0f / c2;
#pragma unroll
    for (int m = -K; m <= K; ++m) {
      if (m < mlo || m > mhi) continue;
      float Yr, Yi;
      const float a = neg ? -(x - (float)m) : (x - (float)m);
      fresnel_bin(a, c1, c2, inv_b, Er, Ei, Yr, Yi);
      if (neg) Yi = -Yi;
      accum(m, Yr, Yi);
    }
  }
}

// Z_c = Re/Im of the per-(SFT, channel) complex term, H_c its <h,h> term (include/sft.h).
template <int KT, int CT>
__device__ __forceinline__ void pair_terms(const KParams &p, const Tmpl &tm, int alpha, const Track &tr,
                                           const float (&us2)[CT], float &zr, float &zi, float &hh) {
  float S1r[CT], S1i[CT], S2[CT];
  float pr, pi_, scale;
  pair_contract<KT, CT>(p, alpha, tr, S1r, S1i, S2, pr, pi_, scale);
  // e^{i phi_a} * (pr + i pi)
  float sp, cp;
  sincospif(2.0f * tr.frac, &sp, &cp);
  const float er = (cp * pr - sp * pi_) * scale * tr.amp;
  const float ei = (cp * pi_ + sp * pr) * scale * tr.amp;
  const float a2 = tr.amp * tr.amp * scale * scale;
  zr = 0.f; zi = 0.f; hh = 0.f;
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    if (c < p.C && us2[c] > 0.f) {
      // response (Eq.(5)-(6) P:80-85 as Lambda z = Re[R z]; DESIGN C3/D4)
      float2 R = tm.AE[c];
      if (p.response == 1) {
        const float2 r = __ldg(p.rtab + (size_t)c * p.n_sft + alpha);
        R = make_float2(tm.AE[c].x * r.x, tm.AE[c].x * r.y);      // AE is real here
      } else if (p.response == 2) {
        const float2 cs = __ldg(p.rtab + (size_t)c * p.n_sft + alpha);
        const float am = fmaf(p.depth, cs.x * tm.cl - cs.y * tm.sl, 1.0f);
        R = make_float2(R.x * am, R.y * am);
      }
      const float gr = R.x * er - R.y * ei, gi = R.x * ei + R.y * er;   // p_c = R * A e^{i phi} pref
      zr += gr * S1r[c] - gi * S1i[c];
      zi += gr * S1i[c] + gi * S1r[c];
      hh += (R.x * R.x + R.y * R.y) * a2 * us2[c] * S2[c];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Main fused kernel.  grid = (template tiles, SFT chunks).  MODE 0: chunk totals only.
// MODE 1 (cumulative): additionally writes chunk-local inclusive prefix sums, transposed through
// shared memory so that global stores are 128-byte rows along the SFT axis.
// ---------------------------------------------------------------------------------------------
template <int KT, int CT, int MODE>
__global__ void __launch_bounds__(TILE) sft_main_kernel(const KParams p) {
  __shared__ float tile_s[MODE == 1 ? (TILE / 32) * 2 * 32 * 33 : 1];
  const long long t = (long long)blockIdx.x * TILE + threadIdx.x;
  const int a0 = blockIdx.y * p.chunk;
  const int a1 = min(a0 + p.chunk, p.n_sft);
  Tmpl tm;
  tmpl_init(p, t, tm);
  double axh = 0.0, ahh = 0.0, axi = 0.0;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float *txh = tile_s + (MODE == 1 ? warp * 2 * 32 * 33 : 0);
  float *thh = txh + (MODE == 1 ? 32 * 33 : 0);

  for (int alpha = a0; alpha < a1; ++alpha) {
    float us2[CT];
    bool any = false;
#pragma unroll
    for (int c = 0; c < CT; ++c) {
      us2[c] = (c < p.C) ? __ldg(p.us2 + (size_t)c * p.n_sft + alpha) : 0.f;
      any |= us2[c] > 0.f;
    }
    Track tr;
    tr.active = false;
    tr.kc = -1;
    if (any || p.kc_out) track_eval(p, tm, alpha, tr);
    if (any && tr.active) {
      float zr, zi, hh;
      pair_terms<KT, CT>(p, tm, alpha, tr, us2, zr, zi, hh);
      axh += (double)zr;
      axi += (double)zi;
      ahh += (double)hh;
    }
    if (p.kc_out && tm.ok) {
#pragma unroll
      for (int c = 0; c < CT; ++c)
        if (c < p.C) p.kc_out[((size_t)t * p.C + c) * p.n_sft + alpha] = (tr.active && us2[c] > 0.f) ? tr.kc : -1;
    }
    if (MODE == 1) {
      const int j = (alpha - a0) & 31;
      txh[lane * 33 + j] = (float)axh;
      thh[lane * 33 + j] = (float)ahh;
      if (j == 31 || alpha == a1 - 1) {
        __syncwarp();
        const int base = alpha - j;
        for (int r = 0; r < 32; ++r) {
          const long long tt = (long long)blockIdx.x * TILE + warp * 32 + r;
          if (tt < p.nT && lane <= j) {
            p.loc_xh[(size_t)tt * p.n_sft + base + lane] = txh[r * 33 + lane];
            p.loc_hh[(size_t)tt * p.n_sft + base + lane] = thh[r * 33 + lane];
          }
        }
        __syncwarp();
      }
    }
  }
  if (tm.ok) {
    double *q = p.part + (size_t)blockIdx.y * 3 * p.nT + t;
    q[0] = axh;
    q[p.nT] = ahh;
    q[2 * p.nT] = axi;
  }
}

// Sum of the chunk totals in fp64, fixed order (deterministic).
__global__ void sft_reduce_kernel(const double *part, long long nT, int n_chunks, double *xh, double *hh,
                                  double *xi) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nT) return;
  double s0 = 0.0, s1 = 0.0, s2 = 0.0;
  for (int c = 0; c < n_chunks; ++c) {
    const double *q = part + (size_t)c * 3 * nT + t;
    s0 += q[0];
    s1 += q[nT];
    s2 += q[2 * nT];
  }
  xh[t] = s0;
  hh[t] = s1;
  if (xi) xi[t] = s2;
}

// Exclusive scan of the chunk totals along the chunk axis, in place, fp64 (the carries).
__global__ void sft_scan_chunks_kernel(double *part, long long nT, int n_chunks) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nT) return;
  double c0 = 0.0, c1 = 0.0;
  for (int c = 0; c < n_chunks; ++c) {
    double *q = part + (size_t)c * 3 * nT + t;
    const double v0 = q[0], v1 = q[nT];
    q[0] = c0;
    q[nT] = c1;
    c0 += v0;
    c1 += v1;
  }
}

// cum = carry (fp64) + chunk-local prefix (fp32);  snr = cum_xh / sqrt(cum_hh)  (0 where cum_hh == 0).
__global__ void sft_fixup_kernel(const double *part, long long nT, int n_sft, int chunk, const float *loc_xh,
                                 const float *loc_hh, float *snr, float *cum_xh, float *cum_hh) {
  for (long long t = blockIdx.y; t < nT; t += gridDim.y) {
    const double *carry = part + t;
    for (int a = blockIdx.x * blockDim.x + threadIdx.x; a < n_sft; a += gridDim.x * blockDim.x) {
      const int ch = a / chunk;
      const size_t i = (size_t)t * n_sft + a;
      const double cx = carry[(size_t)ch * 3 * nT] + (double)loc_xh[i];
      const double chh = carry[(size_t)ch * 3 * nT + nT] + (double)loc_hh[i];
      if (snr) snr[i] = chh > 0.0 ? (float)(cx * rsqrt(chh)) : 0.f;
      if (cum_xh) cum_xh[i] = (float)cx;
      if (cum_hh) cum_hh[i] = (float)chh;
    }
  }
}

// Whitening of one channel at load time (Eq.(15); DESIGN "store").
__global__ void sft_whiten_kernel(const float2 *raw, const double *psd_scale, const double *psd_shape, int n_sft,
                                  int nb, int k_lo, int kv_lo, int kv_hi, double T, double S_ref, float2 *D,
                                  float *us2) {
  const int a = blockIdx.x;
  const double s = psd_scale[a];
  const bool present = isfinite(s) && s > 0.0;
  if (threadIdx.x == 0) us2[a] = present ? (float)(1.0 / s) : 0.f;
  const double pre = present ? 2.0 * sqrt(S_ref / T) / s : 0.0;
  for (int j = threadIdx.x; j < nb; j += blockDim.x) {
    const int k = k_lo + j;
    float2 o = make_float2(0.f, 0.f);
    if (present && k >= kv_lo && k < kv_hi) {
      const double Sk = psd_shape ? psd_shape[j] : 1.0;
      const float2 v = raw[(size_t)a * nb + j];
      const double w = pre / Sk;
      o = make_float2((float)(w * (double)v.x), (float)(-w * (double)v.y));
    }
    D[(size_t)a * nb + j] = o;
  }
}

__global__ void sft_ub2_kernel(const double *psd_shape, int nb, int k_lo, int kv_lo, int kv_hi, double S_ref,
                               float *ub2) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nb) return;
  const int k = k_lo + j;
  const double Sk = psd_shape ? psd_shape[j] : 1.0;
  ub2[j] = (k >= kv_lo && k < kv_hi) ? (float)(S_ref / Sk) : 0.f;
}

// SFT_RESP_ANNUAL: (cos, sin)(2 pi t_a / P + psi_c) per (channel, SFT).
__global__ void sft_annual_table_kernel(int n_sft, double t0, double T, double period, double psi, float2 *out) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n_sft) return;
  double s, c;
  sincos(2.0 * 3.141592653589793 * ((t0 + (double)a * T) / period) + psi, &s, &c);
  out[a] = make_float2((float)c, (float)s);
}

}  // namespace sftk
