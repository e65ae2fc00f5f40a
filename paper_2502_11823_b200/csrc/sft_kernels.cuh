// sft_kernels.cuh - device code of libsft_b200.so (sm_100a).  See include/sft.h for the maths
// and DESIGN.md for the layout; "P:NNN" cites the paper text, "DESIGN xx" a reading in DESIGN.md.
//
// Mapping.  One thread owns one template and walks a chunk of consecutive SFTs; a warp therefore
// holds 32 templates at the SAME SFT, so that (i) every data load is a warp-wide broadcast of the
// same one or two 128-byte lines (templates of a bank tile select the same k_c to within a bin),
// (ii) the branch on the chirp parameter b = fdot T^2 (series order / Fresnel form) is made
// warp-uniform, and (iii) the sum over SFTs needs no cross-lane traffic at all: it is a private
// accumulator per thread (fp32 over 8 SFTs, flushed into fp64).
//
// Scheduling.  The unit of work is (32 templates) x (one chunk of SFTs).  The grid is persistent
// (SM count x resident blocks); every WARP draws work units from one global counter, latest chunks
// (largest b, most expensive) first, so that no SM idles behind a tail of equal-sized blocks.  The
// per-template constants are computed once per call by sft_tmpl_kernel.
//
// Evaluators.  For |b| = |fdot| T^2 <= 1 a template reads pre-contracted data moments from the tables of
// sft_table.cuh (64 or 128 bytes and 19 or 71 packed FMAs per (SFT, channel)); otherwise, or when the plan
// has no tables, the 2K+1 kernel coefficients are evaluated and contracted directly:
//
// Direct inner loop.  The 2K+1 bins of a pair are processed two adjacent bins at a time with the packed
// fp32x2 instructions of sm_100 (FADD2/FMUL2/FFMA2: one issue slot, two lanes).  The store keeps
// the whitened data "pair-planar", {re_j, re_j+1, im_j, im_j+1} per 16 bytes, in two copies (pairs
// starting at even / odd bins), so that ONE aligned 128-bit load delivers both packed operands of a
// bin pair whatever the parity of the window start k_c - K; rows are zero-padded by 2K+2 bins on
// both sides, so no per-bin band-edge test exists.  One MUFU reciprocal serves both bins of a pair
// (1/a = (a-1)/(a(a-1))).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "fresnel_aux_coeffs.h"
#include "sft_table.cuh"

namespace sftk {

constexpr int TILE = 128;            // templates (= threads) per block
constexpr int MAXC = 4;              // SFT_MAX_CHANNELS
constexpr int FLUSH = 8;             // SFTs summed in fp32 before the fp64 accumulators are touched
constexpr double GMSUN_S = 4.925491025543576e-6;   // G Msun / c^3 [s]
constexpr float PI_F = 3.14159265358979f;
// 1.5PN ("tail") coefficients of TaylorT3 in Theta^(-3/8) relative to the leading term: phase -3 pi/4, frequency -3 pi/10
constexpr double C15_PHI = -0.75 * 3.141592653589793, C15_F = -0.3 * 3.141592653589793;
constexpr float INV_2PI_F = 0.15915494309189535f;

// b = fdot T^2 thresholds of the coefficient evaluator (DESIGN "kernel evaluator"): the power
// series in b about the SFT mid-point truncated after order n has error <= (pi b)^(n+1) /
// ((n+1)! 4^(n+1) (2n+3)); the bounds below keep that under 2e-6.
constexpr float B_ORDER1 = 0.0057f;  // |b| <= : order 1
constexpr float B_ORDER2 = 0.056f;   // |b| <= : order 2
constexpr float B_ORDER3 = 0.18f;    // |b| <= : order 3; above: closed Fresnel form

struct KParams {
  int C, n_sft, nb, k_lo, kv_lo, kv_hi, K, PAD, npair;
  int kwin0, jmax;         // window start j0 = k_c - kwin0 in the padded row; in band iff 2 <= j0 <= jmax + 2
  unsigned dstride, cstrideD, cstrideU;   // entries: per channel (n_sft*npair), per copy (C*n_sft*npair), (C*npair)
  int kernel, pn1, response, phase_path;
  double T, t0, f_loT, f_hiT, inv_fref;
  double sigma[MAXC];      // sqrt(T / S_ref,c)
  double chi[MAXC];        // SFT_RESP_ANNUAL response phase per channel
  float depth;
  const float4 *Dp;        // [2][C][n_sft][npair]  {re_j, re_j+1, im_j, im_j+1} of
                           //                        2 conj(x~) sqrt(S_ref) / (sqrt(T) s_a S_k), padded index j = 2i+copy
  const float2 *ubp;       // [2][C][npair]         {u_j, u_j+1}, u = S_ref / S_k (0 for invalid bins)
  const float *us2;        // [C][n_sft]            1 / s_a       (0 for gaps)
  const float2 *rtab;      // [C][n_sft]            TABLE: R_{c,a}; ANNUAL: (cos, sin)(2 pi t_a/P + psi_c)
  const double *params;    // [nT][8]
  const double *td;        // [TD_N][nT]  per-template fp64 constants (sft_tmpl_kernel)
  const float *tf;         // [TF_N][nT]  per-template fp32 constants
  long long nT;
  int chunk, n_chunks;
  int n_tgroups, n_items;  // work units: n_tgroups = ceil(nT/32) template groups x n_chunks
  int *counter;            // work-unit counter (zeroed before every launch): units first_dyn, first_dyn + 1, ... are drawn from it
  int first_dyn;           // = warps of the grid: warp w of the grid starts on unit w without asking (set by launch_variant)
  unsigned long long *path_counts;   // nullable [PATH_N]: active pairs per evaluator path (diagnostic)
  // moment-table evaluator (sft_table.cuh); mtab == nullptr: direct evaluator only
  const float4 *mtab;      // [C][n_sft][n_node][4]   8 complex64 moments per node, node = kcidx * TAB_R + cell
  const float4 *htab;      // [C][n_kc * HTAB_R][4]   <h,h> polynomial per node (tier 2)
  const float4 *htab1;     // [C][n_kc * HT1_R]       compact tier-1 <h,h> node {h_00, h_10, h_20, h_02}
  unsigned h1chan;         // entries of htab1 per channel
  // The moment table is laid out per block of 32 SFT slots (tblk[a >> 5]): rows of W window positions starting at
  // position kb (counted from k_lo - K), so that a bank around a known track needs only the band the track sweeps
  // (sft_plan_set_table_track); without a track every block covers all n_kc positions.
  const int4 *tblk;        // per block {x: float4 index of the block's first row (channel 0), y: kb, z: W, w: float4 per row}
  int banded;              // 0: every block covers all window positions (the in-band test implies the in-table test)
  unsigned mrow0;          // float4 per row of the full (not banded) layout: kernel variants compiled with BAND = false use it
                           // as a constant-bank operand instead of the per-block record
  unsigned mchan;          // float4 entries per channel of mtab; hchan likewise for htab
  unsigned hchan;
  float b_table, b_table2; // B_TABLE, B_TABLE2 if the plan has the tables, else -1 (no |b| qualifies)
  double *part;            // [n_chunks][3][nT] chunk totals (xh, hh, xh_im)
  int *kc_out;             // [nT][C][n_sft] or null
  // cumulative mode (MODE 1): single-pass scan over the SFT axis with decoupled look-back (one work unit = 32 SFT slots)
  float *out_snr, *out_cx, *out_ch;   // [nT][n_sft] outputs, each nullable
  double2 *scanA, *scanP;  // [n_chunks][nT] {xh, hh} + tag: a unit's own totals (aggregate) / totals of all SFTs up to its end (inclusive)
  unsigned epoch;          // 16-bit tag (1 ... 65534) carried by every entry published in this call (scan_publish)
#ifdef SFT_CHECKED
  // checked build (build.py --checked): every indexed global access of the main path is tested against the extent of
  // its buffer (entries, counted in the pointer's element type); the first failing site leaves its code in *chk and the
  // call returns SFT_ECUDA.  The sizes below are those of the allocations in sft_lib.cu, not derived from the indices.
  unsigned *chk;
  unsigned long long n_Dp, n_ubp, n_sl, n_mtab, n_htab, n_htab1, n_tblk, n_out, n_scan, n_part, n_kc;
#endif
};

// SFT_CHK(p, condition, site): no code at all in the product build
#ifdef SFT_CHECKED
#define SFT_CHK(p, cond, site) do { if (!(cond)) atomicCAS((p).chk, 0u, (unsigned)(site)); } while (0)
#define SFT_CHK_TB(p, a) ((unsigned long long)((a) >> 5) < (p).n_tblk ? 0u : atomicCAS((p).chk, 0u, (unsigned)CHK_TBLK))
#else
#define SFT_CHK(p, cond, site) do { } while (0)
#define SFT_CHK_TB(p, a) ((void)0)
#endif
// entries [ptr, ptr + cnt) inside [base, base + n)
#define SFT_CHK_RANGE(p, ptr, cnt, base, n, site) \
  SFT_CHK(p, (unsigned long long)((ptr) - (base)) + (unsigned long long)(cnt) <= (unsigned long long)(n) && (ptr) >= (base), site)
enum ChkSite { CHK_TMPL = 1, CHK_DP, CHK_UBP, CHK_MTAB, CHK_HTAB, CHK_MTAB_FAST, CHK_HTAB1_FAST, CHK_RESP, CHK_US2, CHK_TBLK,
               CHK_SCAN, CHK_OUT, CHK_PART, CHK_KC };

__device__ __forceinline__ float rcp_approx(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float sqrt_approx(float x) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float lg2_approx(float x) {
  float r;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float ex2_approx(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
// (sin, cos)(pi t) for |t| <~ 2 on the MUFU (absolute error ~5e-7)
__device__ __forceinline__ void sincospi_fast(float t, float &s, float &c) {
  const float a = PI_F * t;
  s = __sinf(a);
  c = __cosf(a);
}
__device__ __forceinline__ float2 bc(float v) { return make_float2(v, v); }

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

// Compile-time plan flags of a kernel variant; -1 = read the flag from KParams at run time.
template <int KERNEL_, int PN1_, int RESP_, int KC_, int PHASE_ = 0>
struct Cfg {
  static constexpr int KERNEL = KERNEL_, PN1 = PN1_, RESP = RESP_, KC = KC_, PHASE = PHASE_;
};
template <class CFG> __device__ __forceinline__ int cfg_phase(const KParams &p) { return CFG::PHASE >= 0 ? CFG::PHASE : p.phase_path; }
template <class CFG> __device__ __forceinline__ int cfg_kernel(const KParams &p) { return CFG::KERNEL >= 0 ? CFG::KERNEL : p.kernel; }
// PN order code of the waveform: 0 = 0PN, 1 = 0PN+1PN, 2 = 0PN+1PN+1.5PN (SFT_WF_*)
template <class CFG> __device__ __forceinline__ int cfg_pn1(const KParams &p) { return CFG::PN1 >= 0 ? CFG::PN1 : p.pn1; }
template <class CFG> __device__ __forceinline__ int cfg_resp(const KParams &p) { return CFG::RESP >= 0 ? CFG::RESP : p.response; }

// Per-template constants, fp64 where the phase needs it (the template is "described by 4
// numbers" per SFT; these are the closed-form coefficients of those 4 numbers, DESIGN W1).
// Layout in global memory: structure of arrays, component-major with stride nT.
enum { TD_TAU0 = 0, TD_CTHETA, TD_PHIC, TD_CPHASE, TD_CPHI, TD_CF, TD_F0T, TD_BSCALE, TD_N };
enum { TF_CF = 0, TF_CL, TF_SL, TF_AE, TF_N = TF_AE + 2 * MAXC };

// Double-float ("split fp32") arithmetic for SFT_PHASE_SPLIT32: a value is the unevaluated sum h + l of two
// floats, |l| <= ulp(h)/2 (48-bit significand).  Error-free transformations with explicit rounding intrinsics
// (no contraction).
struct df32 {
  float h, l;
};
__device__ __forceinline__ df32 df_quick(float a, float b) {       // |a| >= |b|
  const float s = __fadd_rn(a, b);
  return {s, __fsub_rn(b, __fsub_rn(s, a))};
}
__device__ __forceinline__ df32 df_two_sum(float a, float b) {
  const float s = __fadd_rn(a, b), bb = __fsub_rn(s, a);
  return {s, __fadd_rn(__fsub_rn(a, __fsub_rn(s, bb)), __fsub_rn(b, bb))};
}
__device__ __forceinline__ df32 df_add(df32 x, df32 y) {
  const df32 s = df_two_sum(x.h, y.h);
  return df_quick(s.h, __fadd_rn(s.l, __fadd_rn(x.l, y.l)));
}
__device__ __forceinline__ df32 df_neg(df32 x) { return {-x.h, -x.l}; }
__device__ __forceinline__ df32 df_mul(df32 x, df32 y) {
  const float ph = __fmul_rn(x.h, y.h);
  float pl = __fmaf_rn(x.h, y.h, -ph);
  pl = __fmaf_rn(x.h, y.l, pl);
  pl = __fmaf_rn(x.l, y.h, pl);
  return df_quick(ph, pl);
}
__device__ __forceinline__ df32 df_mul_f(df32 x, float c) {
  const float ph = __fmul_rn(x.h, c);
  return df_quick(ph, __fmaf_rn(x.l, c, __fmaf_rn(x.h, c, -ph)));
}
__device__ __forceinline__ df32 df_from(double d) {
  const float h = (float)d;
  return {h, (float)(d - (double)h)};
}
// x > y ?
__device__ __forceinline__ bool df_gt(df32 x, df32 y) { return x.h > y.h || (x.h == y.h && x.l > y.l); }
__device__ __forceinline__ bool df_ge(df32 x, df32 y) { return x.h > y.h || (x.h == y.h && x.l >= y.l); }

struct TmplS {           // the fp64 members of Tmpl as double-floats (SFT_PHASE_SPLIT32 only)
  df32 tau0, cTheta, phic_cyc, cphase, cphi, cf, F0T, bscale, T, f_loT, f_hiT;
};

struct Tmpl {
  double tau0, cTheta, phic_cyc, cphase, cphi, cf, F0T, bscale;   // tau0 = t_c - t0
  float cf32, cl, sl;
  float2 AE[MAXC];   // amp (F0/f_ref)^(2/3) sigma_c e^{i(chi_c+beta)}
  TmplS s;
};

#ifndef SFT_MAIN_ONLY      // (the translation units that only instantiate sft_main_kernel skip the small kernels)
// One thread per template, once per call.
__global__ void sft_tmpl_kernel(const KParams p, double *td, float *tf) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t == 0) *p.counter = 0;            // work-unit counter of the main kernel that follows on the stream
  if (t >= p.nT) return;
  const double *row = p.params + t * 8;
  const double mc = row[0], eta = row[1], tc = row[2], phic = row[3], amp = row[4];
  const double lam = row[5], beta = row[6];
  const double M = mc * pow(eta, -0.6) * GMSUN_S;             // total mass [s]
  const double inv2pi = 0.15915494309189535;
  const double cTheta = eta / (5.0 * M);
  const double cf = p.pn1 ? (743.0 / 2688.0 + 11.0 / 32.0 * eta) : 0.0;
  const double F0 = 1.0 / (8.0 * 3.141592653589793 * M);
  const long long n = p.nT;
  td[TD_TAU0 * n + t] = tc - p.t0;
  td[TD_CTHETA * n + t] = cTheta;
  td[TD_PHIC * n + t] = phic * inv2pi;
  td[TD_CPHASE * n + t] = (2.0 / eta) * inv2pi;
  td[TD_CPHI * n + t] = p.pn1 ? (3715.0 / 8064.0 + 55.0 / 96.0 * eta) : 0.0;
  td[TD_CF * n + t] = cf;
  td[TD_F0T * n + t] = F0 * p.T;
  td[TD_BSCALE * n + t] = cTheta * F0 * p.T * p.T;
  const double A0 = amp * cbrt((F0 * p.inv_fref) * (F0 * p.inv_fref));
  double sl, cl;
  sincos(lam, &sl, &cl);
  tf[TF_CF * n + t] = (float)cf;
  tf[TF_CL * n + t] = (float)cl;
  tf[TF_SL * n + t] = (float)sl;
  for (int c = 0; c < MAXC; ++c) {
    float2 ae = make_float2(0.f, 0.f);
    if (c < p.C) {
      double s, co;
      const double ang = (p.response == 2) ? (p.chi[c] + beta) : 0.0;
      sincos(ang, &s, &co);
      const double a = A0 * p.sigma[c];
      ae = make_float2((float)(a * co), (float)(a * s));
    }
    tf[(TF_AE + 2 * c) * n + t] = ae.x;
    tf[(TF_AE + 2 * c + 1) * n + t] = ae.y;
  }
}

#endif  // SFT_MAIN_ONLY

// Lanes beyond the last template run as copies of the last one (so that a ragged last warp, or a bank smaller than a warp, still
// takes the clean-block path); nothing of theirs is ever stored or counted (every output is guarded by t < nT).
template <int CT>
__device__ __forceinline__ void tmpl_load(const KParams &p, long long t, Tmpl &tm) {
  const bool ok = t < p.nT;
  const long long n = p.nT, tt = ok ? t : n - 1;
  const double *d = p.td + tt;
  const float *f = p.tf + tt;
  SFT_CHK(p, tt >= 0 && tt < n, CHK_TMPL);
  tm.tau0 = __ldg(d + TD_TAU0 * n);
  tm.cTheta = __ldg(d + TD_CTHETA * n);
  tm.phic_cyc = __ldg(d + TD_PHIC * n);
  tm.cphase = __ldg(d + TD_CPHASE * n);
  tm.cphi = __ldg(d + TD_CPHI * n);
  tm.cf = __ldg(d + TD_CF * n);
  tm.F0T = __ldg(d + TD_F0T * n);
  tm.bscale = __ldg(d + TD_BSCALE * n);
  tm.cf32 = __ldg(f + TF_CF * n);
  tm.cl = __ldg(f + TF_CL * n);
  tm.sl = __ldg(f + TF_SL * n);
#pragma unroll
  for (int c = 0; c < CT; ++c)
    tm.AE[c] = make_float2(__ldg(f + (TF_AE + 2 * c) * n), __ldg(f + (TF_AE + 2 * c + 1) * n));
  if (p.phase_path == 1) {           // once per work unit: the per-SFT arithmetic then stays off the FP64 pipe
    tm.s.tau0 = df_from(tm.tau0); tm.s.cTheta = df_from(tm.cTheta); tm.s.phic_cyc = df_from(tm.phic_cyc);
    tm.s.cphase = df_from(tm.cphase); tm.s.cphi = df_from(tm.cphi); tm.s.cf = df_from(tm.cf);
    tm.s.F0T = df_from(tm.F0T); tm.s.bscale = df_from(tm.bscale); tm.s.T = df_from(p.T);
    tm.s.f_loT = df_from(p.f_loT); tm.s.f_hiT = df_from(p.f_hiT);
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

// fp64 track, branch-free (so that it can be scheduled into the straight-line code of the bin loop of
// the previous SFT).  tau = t_c - t_a = (t_c - t0) - a T in one fma (t_a differs from the separately
// rounded t0 + a T of P:157 by at most one ulp of t_a, i.e. ~1e-11 s: 1e-9 rad of phase, 1e-13 bins).
// Theta^(-1/8) comes from an fp32 MUFU seed (relative error e ~ 5e-7) refined by one second-order
// Newton step in fp64:  with r = 1 - Theta y^8,  Theta^(-1/8) = y (1-r)^(-1/8)
// = y (1 + r/8 + 9 r^2/128 + O(r^3));  r ~ 8e, so the result is good to ~0.05 (8e)^3 ~ 3e-18 (+ rounding).
// tau <= 0 gives NaNs, which fail every comparison of the activity mask.  Rounding to the nearest
// integer is done by adding 1.5 * 2^52 (|values| < 2^31): k_c = rint(y) equals floor(y + 1/2) except
// for y exactly half-way between two bins, which DESIGN A5 flags as a tie anyway.
constexpr double RND_MAGIC = 6755399441055744.0;   // 1.5 * 2^52

// The same track in double-float arithmetic (SFT_PHASE_SPLIT32): no FP64 instruction per SFT.  Relative
// accuracy ~1e-14 (2^-48 per operation): 1e-8 rad at 1e6 rad of phase, 1e-11 bins.
template <class CFG>
__device__ __forceinline__ void track_eval_split32(const KParams &p, const Tmpl &tm, double dalpha, Track &tr) {
  const TmplS &c = tm.s;
  const float al = (float)dalpha;                                   // SFT index: exact in fp32 (< 2^24)
  const df32 tau = df_add(c.tau0, df_neg(df_mul_f(c.T, al)));
  const df32 theta = df_mul(c.cTheta, tau);
  const float y0 = ex2_approx(-0.125f * lg2_approx(theta.h));
  const df32 y = {y0, 0.f};
  const df32 y2 = df_mul(y, y), y4 = df_mul(y2, y2), y8 = df_mul(y4, y4);
  const df32 one = {1.f, 0.f};
  const df32 r = df_add(one, df_neg(df_mul(theta, y8)));            // ~8e: fp32 accuracy would do, kept in df for the sum
  const float sr = fmaf(r.h, 9.0f / 128.0f, 0.125f) * r.h;          // s = r/8 + 9 r^2/128, |s| ~ 1e-6: fp32 suffices
  const df32 q = df_add(y, df_mul_f(y, sr));                        // Theta^(-1/8), error ~ y * 6e-8 * |s| ~ 1e-13
  const df32 q2 = df_mul(q, q), q3 = df_mul(q2, q), q4 = df_mul(q2, q2), q8 = df_mul(q4, q4), q11 = df_mul(q8, q3);
  const bool pn1 = cfg_pn1<CFG>(p) != 0, pn15 = cfg_pn1<CFG>(p) >= 2;
  df32 ph, fT, b;
  const df32 thq3 = df_mul(theta, q3);
  if (pn1) {
    df32 gp = df_add(one, df_mul(c.cphi, q2)), gf = df_add(one, df_mul(c.cf, q2));
    const df32 k375 = {0.375f, 0.f};
    df32 gb = df_add(k375, df_mul_f(df_mul(c.cf, q2), 0.625f));
    if (pn15) {
      gp = df_add(gp, df_mul(df_from(C15_PHI), q3));
      gf = df_add(gf, df_mul(df_from(C15_F), q3));
      gb = df_add(gb, df_mul(df_from(0.75 * C15_F), q3));
    }
    ph = df_add(c.phic_cyc, df_neg(df_mul(df_mul(c.cphase, thq3), gp)));
    fT = df_mul(df_mul(c.F0T, q3), gf);
    b = df_mul(df_mul(c.bscale, q11), gb);
  } else {
    ph = df_add(c.phic_cyc, df_neg(df_mul(c.cphase, thq3)));
    fT = df_mul(c.F0T, q3);
    b = df_mul_f(df_mul(c.bscale, q11), 0.375f);
  }
  const df32 yy = (cfg_kernel<CFG>(p) == 1) ? df_add(fT, df_mul_f(b, 0.5f)) : fT;
  // k_c = rint(yy): round the high part, fix up with the rest (|rest| can exceed 1/2 by the low part only)
  float kf = rintf(yy.h);
  float rest = __fadd_rn(__fsub_rn(yy.h, kf), yy.l);
  if (rest > 0.5f) { kf += 1.0f; rest -= 1.0f; }
  if (rest < -0.5f) { kf -= 1.0f; rest += 1.0f; }
  tr.active = df_gt(tau, c.T) && df_ge(fT, c.f_loT) && df_ge(c.f_hiT, df_add(fT, b));
  tr.kc = (int)kf;
  const df32 xd = df_add(fT, {-kf, 0.f});
  tr.x = xd.h;
  tr.b = b.h;
  const float pk = rintf(ph.h);
  float fr = __fadd_rn(__fsub_rn(ph.h, pk), ph.l);
  tr.frac = fr - rintf(fr);
  const float q2f = y0 * y0;
  float a = q2f;
  if (pn1) a *= ex2_approx((2.0f / 3.0f) * lg2_approx(fmaf(tm.cf32, q2f, 1.0f) + (pn15 ? (float)C15_F * (q2f * y0) : 0.f)));
  tr.amp = a;
}

template <class CFG>
__device__ __forceinline__ void track_eval_fp64(const KParams &p, const Tmpl &tm, double dalpha, Track &tr);

template <class CFG>
__device__ __forceinline__ void track_eval(const KParams &p, const Tmpl &tm, double dalpha, Track &tr) {
  if (cfg_phase<CFG>(p) == 1) track_eval_split32<CFG>(p, tm, dalpha, tr);
  else track_eval_fp64<CFG>(p, tm, dalpha, tr);
}

template <class CFG>
__device__ __forceinline__ void track_eval_fp64(const KParams &p, const Tmpl &tm, double dalpha, Track &tr) {
  const double tau = fma(-dalpha, p.T, tm.tau0);
  const double theta = tm.cTheta * tau;
  const float y0 = ex2_approx(-0.125f * lg2_approx((float)theta));
  const double y = (double)y0;
  const double y2 = y * y, y4 = y2 * y2, y8 = y4 * y4;
  const double r = fma(-theta, y8, 1.0);
  const double s = fma(r, 9.0 / 128.0, 0.125) * r;
  const double q = fma(y, s, y);                  // Theta^(-1/8)
  const double q2 = q * q, q3 = q2 * q, q4 = q2 * q2, q8 = q4 * q4;
  const bool pn1 = cfg_pn1<CFG>(p) != 0, pn15 = cfg_pn1<CFG>(p) >= 2;
  double ph, fT, b;
  if (pn1) {
    double gp = fma(tm.cphi, q2, 1.0), gf = fma(tm.cf, q2, 1.0), gb = fma(0.625 * tm.cf, q2, 0.375);
    if (pn15) {                                     // 1.5PN tail terms, relative order Theta^(-3/8) = q^3
      gp = fma(C15_PHI, q3, gp);
      gf = fma(C15_F, q3, gf);
      gb = fma(0.75 * C15_F, q3, gb);
    }
    ph = fma(-tm.cphase * (theta * q3), gp, tm.phic_cyc);   // cycles
    fT = tm.F0T * q3 * gf;
    b = tm.bscale * (q8 * q3) * gb;
  } else {
    ph = fma(-tm.cphase, theta * q3, tm.phic_cyc);
    fT = tm.F0T * q3;
    b = (0.375 * tm.bscale) * (q8 * q3);
  }
  const double yy = (cfg_kernel<CFG>(p) == 1) ? fma(0.5, b, fT) : fT;   // Fresnel: centre of the swept band
  const double kr = yy + RND_MAGIC;                // f_hiT is clamped by the host: active => |yy| < 2^30
  const double pr = ph + RND_MAGIC;
  tr.active = (tau > p.T) && (fT >= p.f_loT) && (fT + b <= p.f_hiT);
  tr.kc = __double2loint(kr);
  tr.x = (float)(fT - (kr - RND_MAGIC));
  tr.b = (float)b;
  tr.frac = (float)(ph - (pr - RND_MAGIC));
  // amplitude (f_a/F0)^(2/3) = q^2 (1 + cf q^2)^(2/3): the seed is good enough (1e-6 relative)
  const float q2f = y0 * y0;
  float a = q2f;
  if (pn1) a *= ex2_approx((2.0f / 3.0f) * lg2_approx(fmaf(tm.cf32, q2f, 1.0f) + (pn15 ? (float)C15_F * (q2f * y0) : 0.f)));
  tr.amp = a;
}

// ---------------------------------------------------------------------------------------------
// Coefficient evaluator.  F(x-m, b) = e^{i pi (x + b/4)} J_m with (DESIGN "kernel evaluator")
//   J_m = (-1)^m int_{-1/2}^{1/2} e^{i (w v + pi b v^2)} dv,  w = 2 pi a',  a' = x + b/2 - m
//       = sum_n (i pi b)^n / n! r_2n(a'),   r_j = (-1)^m int v^j e^{i w v} dv,
// expanded about the SFT mid-point.  Far bins (m != 0, |a'| >= 1/2) use the forward recurrence
//   r_0 = 2 S w', q_1 = (r_0 - C) w', r_2 = (S/2 - 2 q_1) w', q_3 = (3 r_2 - C/4) w', ...   w' = 1/w,
// with S = sin(pi xp), C = cos(pi xp), xp = x + b/2 (the (-1)^m of sin/cos(pi a') cancels the one in
// J_m).  The central bin (m = 0, |a'| <= 1/2 by construction of k_c, DESIGN A5) uses the Taylor
// series in z = (pi a')^2.  b = 0 is the Dirichlet kernel e^{i pi a} sinc(a), Eq.(B2) P:451.
// ---------------------------------------------------------------------------------------------
// All evaluators below return J^ = 2 pi J (the common factor kappa = 1/(2 pi) of the far recurrence is
// applied once per (template, SFT) instead of once per bin): with u = 1/a' and X^ = X / kappa,
//   r^_0 = 2 S u,  q^_1 = (kappa r^_0 - C) u,  r^_2 = (S/2 - 2 kappa q^_1) u,  q^_3 = (3 kappa r^_2 - C/4) u, ...
template <int ORD>
struct SeriesK {           // per-(template, SFT) constants, broadcast into both packed lanes
  float2 S2, mC, c_i0, c_i1, c_i2;      // 2S, -C, and for order 1:  J^_i = (c_i0 + (c_i1 + c_i2 u) u) u
  float2 Sh, mC4, S8, mC16, S32;        // higher orders
  float2 pb, mpb2h, mpb3s;              // pi b, -(pi b)^2/2, -(pi b)^3/6
  float pbs;
};

template <int ORD>
__device__ __forceinline__ void series_setup(float xp, float b, SeriesK<ORD> &k) {
  float S, C;
  sincospi_fast(xp, S, C);
  const float pb = PI_F * b;
  k.pbs = pb;
  k.S2 = bc(2.0f * S);
  k.mC = bc(-C);
  if (ORD == 1) {       // J^_i = pi b r^_2 = pi b (S/2 - 2 kappa (2 kappa S u - C) u) u, expanded in u
    k.c_i0 = bc(0.5f * pb * S);
    k.c_i1 = bc(2.0f * INV_2PI_F * pb * C);
    k.c_i2 = bc(-4.0f * INV_2PI_F * INV_2PI_F * pb * S);
  }
  if (ORD >= 2) {
    k.Sh = bc(0.5f * S);
    k.mC4 = bc(-0.25f * C);
    k.S8 = bc(0.125f * S);
    k.pb = bc(pb);
    k.mpb2h = bc(-0.5f * pb * pb);
  }
  if (ORD >= 3) {
    k.mC16 = bc(-0.0625f * C);
    k.S32 = bc(0.03125f * S);
    k.mpb3s = bc(-(1.0f / 6.0f) * pb * pb * pb);
  }
}

// two far bins at once; u = {1/a_lo, 1/a_hi}
template <int ORD>
__device__ __forceinline__ void series_far2(const SeriesK<ORD> &k, float2 u, float2 &Jr, float2 &Ji) {
  const float2 r0 = __fmul2_rn(k.S2, u);
  Jr = r0;
  if (ORD == 0) {
    Ji = make_float2(0.f, 0.f);
  } else {
    if (ORD == 1) {
      Ji = __fmul2_rn(__ffma2_rn(__ffma2_rn(k.c_i2, u, k.c_i1), u, k.c_i0), u);
    } else {
      const float2 q1 = __fmul2_rn(__ffma2_rn(bc(INV_2PI_F), r0, k.mC), u);
      const float2 r2 = __fmul2_rn(__ffma2_rn(bc(-2.0f * INV_2PI_F), q1, k.Sh), u);
      const float2 q3 = __fmul2_rn(__ffma2_rn(bc(3.0f * INV_2PI_F), r2, k.mC4), u);
      const float2 r4 = __fmul2_rn(__ffma2_rn(bc(-4.0f * INV_2PI_F), q3, k.S8), u);
      Jr = __ffma2_rn(k.mpb2h, r4, r0);
      Ji = __fmul2_rn(k.pb, r2);
      if (ORD >= 3) {
        const float2 q5 = __fmul2_rn(__ffma2_rn(bc(5.0f * INV_2PI_F), r4, k.mC16), u);
        const float2 r6 = __fmul2_rn(__ffma2_rn(bc(-6.0f * INV_2PI_F), q5, k.S32), u);
        Ji = __ffma2_rn(k.mpb3s, r6, Ji);
      }
    }
  }
}

// {1/a, 1/b} with one MUFU reciprocal
__device__ __forceinline__ float2 rcp2(float a, float b) {
  const float rp = rcp_approx(a * b);
  return make_float2(b * rp, a * rp);
}

// {1/a, 1/(a-1)} with one MUFU reciprocal and one rounding per result:  a (a-1) = fma(a, a, -a)
__device__ __forceinline__ float2 rcp2_adj(float a) {
  const float rp = rcp_approx(fmaf(a, a, -a));
  return make_float2(fmaf(a, rp, -rp), a * rp);
}

// Taylor coefficients of 2 pi r_2n(a') = 2 pi 4^-n sum_p (-1)^p z^p / ((2p)! (2n+2p+1)),  z = (pi a')^2 <= (pi/2)^2;
// 7 terms: truncation < 5e-10 (relative to r_0 <= 1).  Packed as {r_0, r_2} and {r_4, r_6}.
__device__ __forceinline__ constexpr float tay_c(int n, int pp) {
  double f = 1.0;
  for (int i = 2; i <= 2 * pp; ++i) f *= (double)i;
  double s = (pp & 1) ? -1.0 : 1.0;
  double four = 1.0;
  for (int i = 0; i < n; ++i) four *= 4.0;
  return (float)(6.283185307179586 * s / (f * (double)(2 * n + 2 * pp + 1) * four));
}

template <int N>
__device__ __forceinline__ float tay_poly(float z) {      // scalar FFMAs with immediate coefficients
  float r = tay_c(N, 6);
#pragma unroll
  for (int pp = 5; pp >= 0; --pp) r = fmaf(r, z, tay_c(N, pp));
  return r;
}

template <int ORD>
__device__ __forceinline__ void series_central(const SeriesK<ORD> &k, float a, float &Jr, float &Ji) {
  const float t = PI_F * a;
  const float z = t * t;
  Jr = tay_poly<0>(z);                    // r^_0
  Ji = 0.f;
  if (ORD >= 1) Ji = k.pbs * tay_poly<1>(z);             // pi b r^_2
  if (ORD >= 2) Jr = fmaf(-0.5f * k.pbs * k.pbs, tay_poly<2>(z), Jr);
  if (ORD >= 3) Ji = fmaf(-(1.0f / 6.0f) * k.pbs * k.pbs * k.pbs, tay_poly<3>(z), Ji);
}

// Closed Fresnel form (Eq.(29)-(30) P:219-226) rewritten with the auxiliary functions so that the
// large phase pi a^2/b cancels analytically (DESIGN "kernel evaluator"):  with l = a sqrt(2/b),
// u = l + sqrt(2b), w(t) = g(t) + i f(t), E = e^{i pi (2x+b)},
//   sqrt(2b) F(a,b) = sgn(l) w(|l|) - E sgn(u) w(|u|) + [l < 0 <= u] (1+i) e^{-i pi a^2/b}.
struct FresK {
  float c1, c2, inv_b, Er, Ei, xs;
  bool neg;
};
__device__ __forceinline__ void fresnel_bin(const FresK &k, int m, float &Yr, float &Yi) {
  // b < 0: F(a,-|b|) = conj F(-a,|b|)  (DESIGN A10)
  const float a = k.neg ? -(k.xs - (float)m) : (k.xs - (float)m);
  const float l = a * k.c1;
  const float u = l + k.c2;
  float gl, fl, gu, fu;
  fresnel_w(fabsf(l), gl, fl);
  fresnel_w(fabsf(u), gu, fu);
  const float sl = (l >= 0.f) ? 1.f : -1.f;
  const float su = (u >= 0.f) ? 1.f : -1.f;
  const float er = k.Er * gu - k.Ei * fu;       // E * w(|u|)
  const float ei = k.Er * fu + k.Ei * gu;
  Yr = sl * gl - su * er;
  Yi = sl * fl - su * ei;
  if (l < 0.f && u >= 0.f) {
    float s, c;
    sincospif(a * a * k.inv_b, &s, &c);     // e^{-i pi a^2/b} = c - i s ;  (1+i)(c - i s) = (c+s) + i(c-s)
    Yr += c + s;
    Yi += c - s;
  }
  if (k.neg) Yi = -Yi;
}

// Per-channel packed accumulators of the contraction over the bins of one (template, SFT):
//   A = sum Dre J_r,  B = sum Dim J_i,  I = sum (Dre J_i + Dim J_r),  W = sum u |J|^2   (lane = bin parity)
struct Acc {
  float2 A, B, I, W;
};

// Where the window of one (template, SFT) sits in the pair-planar store.  j0 = padded index of bin
// m = -K; copy (j0 & 1) holds the pairs starting at even window offsets, the other copy those starting
// at odd offsets; `row`/`urow` point at copy 0 of the SFT's row (channel 0).
struct Win {
  const float4 *dE, *dO;    // entry of window offset i: even i -> dE[i/2], odd i -> dO[(i-1)/2]
  const float2 *uE, *uO;
};
__device__ __forceinline__ void win_init(const KParams &p, const float4 *row, int j0, Win &w) {
  const unsigned cp = (unsigned)j0 & 1u, eE = (unsigned)j0 >> 1, eO = (unsigned)(j0 + 1) >> 1;
  w.dE = row + (cp * p.cstrideD + eE);
  w.dO = row + ((cp ^ 1u) * p.cstrideD + eO);
  w.uE = p.ubp + (cp * p.cstrideU + eE);
  w.uO = p.ubp + ((cp ^ 1u) * p.cstrideU + eO);
}

// pair of adjacent bins at window offsets (i, i+1)
template <int CT>
__device__ __forceinline__ void mac_pair(const KParams &p, const Win &w, int i, float2 Jr, float2 Ji, Acc (&acc)[CT]) {
  const float4 *dp = (i & 1) ? w.dO + (i >> 1) : w.dE + (i >> 1);
  const float2 *up = (i & 1) ? w.uO + (i >> 1) : w.uE + (i >> 1);
  const float2 mag = __ffma2_rn(Ji, Ji, __fmul2_rn(Jr, Jr));
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    SFT_CHK_RANGE(p, dp + c * p.dstride, 1, p.Dp, p.n_Dp, CHK_DP);
    SFT_CHK_RANGE(p, up + c * p.npair, 1, p.ubp, p.n_ubp, CHK_UBP);
    const float4 d = __ldg(dp + c * p.dstride);
    const float2 u = __ldg(up + c * p.npair);
    const float2 dre = make_float2(d.x, d.y), dim = make_float2(d.z, d.w);
    acc[c].A = __ffma2_rn(dre, Jr, acc[c].A);
    acc[c].B = __ffma2_rn(dim, Ji, acc[c].B);
    acc[c].I = __ffma2_rn(dre, Ji, acc[c].I);
    acc[c].I = __ffma2_rn(dim, Jr, acc[c].I);
    acc[c].W = __ffma2_rn(u, mag, acc[c].W);
  }
}

// one bin at window offset i (scalar; accumulates into the lo lanes)
template <int CT>
__device__ __forceinline__ void mac_single(const KParams &p, const Win &w, int i, float Jr, float Ji, Acc (&acc)[CT]) {
  const float4 *dp = (i & 1) ? w.dO + (i >> 1) : w.dE + (i >> 1);
  const float2 *up = (i & 1) ? w.uO + (i >> 1) : w.uE + (i >> 1);
  const float mag = fmaf(Ji, Ji, Jr * Jr);
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    SFT_CHK_RANGE(p, dp + c * p.dstride, 1, p.Dp, p.n_Dp, CHK_DP);
    SFT_CHK_RANGE(p, up + c * p.npair, 1, p.ubp, p.n_ubp, CHK_UBP);
    const float4 d = __ldg(dp + c * p.dstride);
    const float2 u = __ldg(up + c * p.npair);
    acc[c].A.x = fmaf(d.x, Jr, acc[c].A.x);
    acc[c].B.x = fmaf(d.z, Ji, acc[c].B.x);
    acc[c].I.x = fmaf(d.x, Ji, acc[c].I.x);
    acc[c].I.x = fmaf(d.z, Jr, acc[c].I.x);
    acc[c].W.x = fmaf(u.x, mag, acc[c].W.x);
  }
}

// Series path of one (template, SFT).  The 2K far bins are taken two adjacent bins at a time -
// (-K,-K+1), ..., (-2,-1) on the low side, (1,2), ..., (K-1,K) on the high side (for odd K the bins
// -1 and +1 are left over and evaluated as one non-adjacent pair) - and the central bin m = 0 alone.
// `nxt` = track of the NEXT SFT: it does not depend on anything here and sits in this straight-line
// code so that its fp64 dependency chain is issued between the fp32 work of the bin loop.
template <int ORD, int KT, int CT, class CFG>
__device__ __forceinline__ void series_pairs(const KParams &p, const Tmpl &tm, double dnext, Track &nxt, float xp, float b,
                                             const Win &w, Acc (&acc)[CT]) {
  const int K = KT > 0 ? KT : p.K;
  SeriesK<ORD> k;
  series_setup<ORD>(xp, b, k);
  track_eval<CFG>(p, tm, dnext, nxt);
  const int odd = K & 1, half = K >> 1;
  const float aN = xp + (float)K;              // a' of m = -K
  const float aP = xp - (float)(1 + odd);      // a' of the first high-side pair's lo bin
#pragma unroll
  for (int q = 0; q < half; ++q) {
    float2 Jr, Ji;
    series_far2<ORD>(k, rcp2_adj(aN - (float)(2 * q)), Jr, Ji);
    mac_pair<CT>(p, w, 2 * q, Jr, Ji, acc);
  }
  {
    float c_r, c_i;
    series_central<ORD>(k, xp, c_r, c_i);
    mac_single<CT>(p, w, K, c_r, c_i, acc);
  }
  if (odd) {
    float2 Jr, Ji;
    series_far2<ORD>(k, rcp2(xp + 1.0f, xp - 1.0f), Jr, Ji);
    mac_single<CT>(p, w, K - 1, Jr.x, Ji.x, acc);
    mac_single<CT>(p, w, K + 1, Jr.y, Ji.y, acc);
  }
#pragma unroll
  for (int q = 0; q < half; ++q) {
    float2 Jr, Ji;
    series_far2<ORD>(k, rcp2_adj(aP - (float)(2 * q)), Jr, Ji);
    mac_pair<CT>(p, w, K + 1 + odd + 2 * q, Jr, Ji, acc);
  }
}

template <int KT, int CT, class CFG>
__device__ __forceinline__ void fresnel_pairs(const KParams &p, const Tmpl &tm, double dnext, Track &nxt, float x, float b,
                                              const Win &w, Acc (&acc)[CT], float &scale) {
  const int K = KT > 0 ? KT : p.K;
  track_eval<CFG>(p, tm, dnext, nxt);
  FresK k;
  k.neg = b < 0.f;
  const float ab = fabsf(b);
  k.c1 = sqrtf(2.0f / ab);
  k.c2 = sqrtf(2.0f * ab);
  k.inv_b = 1.0f / ab;
  k.xs = x;
  const float xs = k.neg ? -x : x;
  sincospif(fmaf(2.0f, xs, ab), &k.Ei, &k.Er);
  scale = 1.0f / k.c2;
#pragma unroll 1
  for (int q = 0; q <= K; ++q) {
    float2 Jr, Ji;
    const int m_lo = -K + 2 * q;
    fresnel_bin(k, m_lo, Jr.x, Ji.x);
    if (m_lo + 1 > K) { Jr.y = 0.f; Ji.y = 0.f; }
    else fresnel_bin(k, m_lo + 1, Jr.y, Ji.y);
    mac_pair<CT>(p, w, 2 * q, Jr, Ji, acc);
  }
}

// Evaluator paths (warp-uniform): series order 0..3, closed Fresnel form.
enum { PATH_ORD0 = 0, PATH_ORD1, PATH_ORD2, PATH_ORD3, PATH_FRESNEL, PATH_TABLE, PATH_TABLE2, PATH_N };

__device__ __forceinline__ int path_of(float bmax, bool table) {
  if (table && bmax <= B_TABLE) return PATH_TABLE;   // same tests as pair_terms
  if (table && bmax <= B_TABLE2) return PATH_TABLE2;
  return bmax == 0.f ? PATH_ORD0 : bmax <= B_ORDER1 ? PATH_ORD1 : bmax <= B_ORDER2 ? PATH_ORD2 : bmax <= B_ORDER3 ? PATH_ORD3
                                                                                                               : PATH_FRESNEL;
}

// X + i s Y for complex X, Y held as (re, im) pairs: one packed FMA (swapped, lane-negated operand)
__device__ __forceinline__ float2 cstep(float2 X, float s, float2 Y) {
  return __ffma2_rn(make_float2(-Y.y, Y.x), make_float2(s, s), X);
}

// Moment-table evaluator of one (template, SFT): S1 = sum_m D J_m and S2 = sum_m u |J_m|^2 from the tables
// of sft_table.cuh (true J, no 2 pi).  `kcidx` = k_c - (k_lo - K), already clamped to the table;
// `Mrow` = row of SFT alpha, channel 0.  TIER 1: moments q <= 7, H to beta^2 (|b| <= B_TABLE); TIER 2: q <= 15,
// H to beta^6 (|b| <= B_TABLE2).  Also evaluates the track of the next SFT (see series_pairs).
template <int CT, int TIER>
struct TableData {
  static constexpr int Q = TIER == 1 ? TAB_Q1 : TAB_Q;          // highest moment
  static constexpr int NL = (Q + 1) / 2;                         // float4 loads of moments per channel
  static constexpr int NHB = HTAB_NB;                            // powers of beta^2 in H (tier 2)
  static constexpr int NHL = TIER == 1 ? 1 : (NHB * (HTAB_P + 1) + 3) / 4;   // float4 loads of H coefficients (tier 1: the compact node)
  float4 Mq[CT][NL], Hq[CT][NHL];
  float a, aH, be;
};

// node look-up and loads
template <int CT, int TIER>
__device__ __forceinline__ void table_load(const KParams &p, float xp, float b, int kcidx, int kb, const float4 *Mrow,
                                           TableData<CT, TIER> &d) {
  // node of the <h,h> table: cellH = floor((xp + 1/2) HTAB_R) by the 1.5 * 2^23 rounding trick, clamped (xp = 1/2
  // exactly, NaN lanes); the data-moment node is cellH >> HTAB_SHIFT.  The offset HTAB_R/2 - 1/2 must be added
  // BEFORE the magic constant: 31.5 + 1.5 * 2^23 is not representable (ulp 1) and would turn the floor into a round-to-
  // nearest, i.e. nodes half a cell off.  (At an exact cell edge the rounding may pick either neighbour: same bound.)
  constexpr float RM = 12582912.0f;
  constexpr int HR = TIER == 1 ? HT1_R : HTAB_R, HS = TIER == 1 ? HT1_SHIFT : HTAB_SHIFT;   // tier 1: compact node on the finer grid
  float cm = fmaf(xp, (float)HR, 0.5f * HR - 0.5f) + RM;
  cm = fminf(fmaxf(cm, RM), RM + (float)(HR - 1));
  const int cellH = __float_as_int(cm) & (HR - 1);
  const int cell = cellH >> HS;
  const float cHf = cm - RM;                                   // (float)cellH
  const float4 *mp = Mrow + (unsigned)((kcidx - kb) * TAB_R + cell) * (unsigned)((TAB_Q + 1) / 2);    // row of the block: positions kb ...
  const float4 *hp = TIER == 1 ? p.htab1 + (unsigned)(kcidx * HT1_R + cellH)
                               : p.htab + (unsigned)(kcidx * HTAB_R + cellH) * (unsigned)(HTAB_W / 4);
  const unsigned hch = TIER == 1 ? p.h1chan : p.hchan;
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    SFT_CHK_RANGE(p, mp + c * p.mchan, (TableData<CT, TIER>::NL), p.mtab, p.n_mtab, CHK_MTAB);
    SFT_CHK_RANGE(p, hp + c * hch, (TableData<CT, TIER>::NHL), TIER == 1 ? p.htab1 : p.htab, TIER == 1 ? p.n_htab1 : p.n_htab, CHK_HTAB);
#pragma unroll
    for (int i = 0; i < TableData<CT, TIER>::NL; ++i) d.Mq[c][i] = __ldg(mp + c * p.mchan + i);
#pragma unroll
    for (int i = 0; i < TableData<CT, TIER>::NHL; ++i) d.Hq[c][i] = __ldg(hp + c * hch + i);
  }
  // a = 2 pi (xp - node centre):  centre_H = (cellH + 1/2)/HTAB_R - 1/2,  centre_M = (cell + 1/2)/TAB_R - 1/2
  d.aH = fmaf(cHf, -(2.0f * PI_F) / HR, fmaf(xp, 2.0f * PI_F, (2.0f * PI_F) * (0.5f - 0.5f / HR)));
  d.a = fmaf((float)cell, -(2.0f * PI_F) / TAB_R, fmaf(xp, 2.0f * PI_F, (2.0f * PI_F) * (0.5f - 0.5f / TAB_R)));
  d.be = PI_F * b;
}

// the two Horner evaluations
template <int CT, int TIER>
__device__ __forceinline__ void table_math(const TableData<CT, TIER> &d, float (&s1r)[CT], float (&s1i)[CT], float (&s2)[CT]) {
  constexpr int Q = TableData<CT, TIER>::Q, NHB = TableData<CT, TIER>::NHB;
  const float a = d.a, aH = d.aH, be = d.be;
  float nb_[Q / 2 + 1], na_[Q + 1];                       // beta / k, a / k
#pragma unroll
  for (int k = 1; k <= Q / 2; ++k) nb_[k] = be * (1.0f / (float)k);
#pragma unroll
  for (int k = 1; k <= Q; ++k) na_[k] = a * (1.0f / (float)k);
  const float be2 = be * be;
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    float2 M[Q + 1];
#pragma unroll
    for (int q = 0; q <= Q; ++q)
      M[q] = (q & 1) ? make_float2(d.Mq[c][q >> 1].z, d.Mq[c][q >> 1].w) : make_float2(d.Mq[c][q >> 1].x, d.Mq[c][q >> 1].y);
    // S1 = sum_p (i a)^p / p! L_p,  L_p = sum_n (i beta)^n / n! M_{p+2n}: both by Horner, one packed FMA per step
    float2 S = make_float2(0.f, 0.f);
#pragma unroll
    for (int pq = Q; pq >= 0; --pq) {
      const int nmax = (Q - pq) / 2;
      float2 L = M[pq + 2 * nmax];
#pragma unroll
      for (int n = nmax; n >= 1; --n) L = cstep(M[pq + 2 * (n - 1)], nb_[n], L);
      S = pq == Q ? L : cstep(L, na_[pq + 1], S);
    }
    s1r[c] = S.x;
    s1i[c] = S.y;
    // H = sum_P aH^P sum_N beta^(2N) h_{P,2N};  floats: [N][P], P fastest (tier 1: the compact node {h_00, h_10, h_20, h_02})
    const float *hf = (const float *)&d.Hq[c][0];
    float h = 0.f;
    if (TIER == 1) {
      h = fmaf(be2, hf[3], fmaf(fmaf(hf[2], aH, hf[1]), aH, hf[0]));
    } else {
#pragma unroll
      for (int P = HTAB_P; P >= 0; --P) {
        float g = hf[(NHB - 1) * (HTAB_P + 1) + P];
#pragma unroll
        for (int N = NHB - 2; N >= 0; --N) g = fmaf(g, be2, hf[N * (HTAB_P + 1) + P]);
        h = P == HTAB_P ? g : fmaf(h, aH, g);
      }
    }
    s2[c] = h;
  }
}

// table_math for two independent (template, SFT) streams with every Horner step issued for both in turn, so that the
// dependent chains of one fill the latency of the other without relying on the scheduler's window.
template <int CT, int TIER>
__device__ __forceinline__ void table_math2(const TableData<CT, TIER> &dA, const TableData<CT, TIER> &dB, float (&s1rA)[CT],
                                            float (&s1iA)[CT], float (&s2A)[CT], float (&s1rB)[CT], float (&s1iB)[CT],
                                            float (&s2B)[CT]) {
  constexpr int Q = TableData<CT, TIER>::Q, NHB = TableData<CT, TIER>::NHB;
  float nbA[Q / 2 + 1], naA[Q + 1], nbB[Q / 2 + 1], naB[Q + 1];
#pragma unroll
  for (int k = 1; k <= Q / 2; ++k) { nbA[k] = dA.be * (1.0f / (float)k); nbB[k] = dB.be * (1.0f / (float)k); }
#pragma unroll
  for (int k = 1; k <= Q; ++k) { naA[k] = dA.a * (1.0f / (float)k); naB[k] = dB.a * (1.0f / (float)k); }
  const float be2A = dA.be * dA.be, be2B = dB.be * dB.be;
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    float2 MA[Q + 1], MB[Q + 1];
#pragma unroll
    for (int q = 0; q <= Q; ++q) {
      MA[q] = (q & 1) ? make_float2(dA.Mq[c][q >> 1].z, dA.Mq[c][q >> 1].w) : make_float2(dA.Mq[c][q >> 1].x, dA.Mq[c][q >> 1].y);
      MB[q] = (q & 1) ? make_float2(dB.Mq[c][q >> 1].z, dB.Mq[c][q >> 1].w) : make_float2(dB.Mq[c][q >> 1].x, dB.Mq[c][q >> 1].y);
    }
    float2 SA = make_float2(0.f, 0.f), SB = SA;
#pragma unroll
    for (int pq = Q; pq >= 0; --pq) {
      const int nmax = (Q - pq) / 2;
      float2 LA = MA[pq + 2 * nmax], LB = MB[pq + 2 * nmax];
#pragma unroll
      for (int n = nmax; n >= 1; --n) {
        LA = cstep(MA[pq + 2 * (n - 1)], nbA[n], LA);
        LB = cstep(MB[pq + 2 * (n - 1)], nbB[n], LB);
      }
      SA = pq == Q ? LA : cstep(LA, naA[pq + 1], SA);
      SB = pq == Q ? LB : cstep(LB, naB[pq + 1], SB);
    }
    s1rA[c] = SA.x; s1iA[c] = SA.y;
    s1rB[c] = SB.x; s1iB[c] = SB.y;
    const float *hA = (const float *)&dA.Hq[c][0], *hB = (const float *)&dB.Hq[c][0];
    float ha = 0.f, hb = 0.f;
    if (TIER == 1) {
      ha = fmaf(be2A, hA[3], fmaf(fmaf(hA[2], dA.aH, hA[1]), dA.aH, hA[0]));
      hb = fmaf(be2B, hB[3], fmaf(fmaf(hB[2], dB.aH, hB[1]), dB.aH, hB[0]));
    } else {
#pragma unroll
      for (int P = HTAB_P; P >= 0; --P) {
        float gA = hA[(NHB - 1) * (HTAB_P + 1) + P], gB = hB[(NHB - 1) * (HTAB_P + 1) + P];
#pragma unroll
        for (int N = NHB - 2; N >= 0; --N) {
          gA = fmaf(gA, be2A, hA[N * (HTAB_P + 1) + P]);
          gB = fmaf(gB, be2B, hB[N * (HTAB_P + 1) + P]);
        }
        ha = P == HTAB_P ? gA : fmaf(ha, dA.aH, gA);
        hb = P == HTAB_P ? gB : fmaf(hb, dB.aH, gB);
      }
    }
    s2A[c] = ha;
    s2B[c] = hb;
  }
}

template <int CT, class CFG, int TIER>
__device__ __forceinline__ void table_eval(const KParams &p, const Tmpl &tm, double dnext, Track &nxt, float xp, float b,
                                           int kcidx, int kb, const float4 *Mrow, float (&s1r)[CT], float (&s1i)[CT],
                                           float (&s2)[CT]) {
  TableData<CT, TIER> d;
  table_load<CT, TIER>(p, xp, b, kcidx, kb, Mrow, d);
  track_eval<CFG>(p, tm, dnext, nxt);
  table_math<CT, TIER>(d, s1r, s1i, s2);
}

// Phase, amplitude, response and noise weight applied to the contracted sums of one (template, SFT).
// F-statistic variant (`fq` != nullptr, MODE 2 of the main kernel; Eq.(10)-(13) P:107-122): the plan's response table holds the
// antenna-pattern functions (a, b)_{c,a}; with W = A e^{i phi} sum_k conj(x~) F / S and H = A^2 sum_k |F|^2 / S of the unit
// response, the four basis waveforms h_nu = A [a cos, b cos, a sin, b sin](phi) = Re[(a, b, -i a, -i b) A e^{i phi}] give
//   ([x,h_0]) + i ([x,h_2]) = sum a W,   ([x,h_1]) + i ([x,h_3]) = sum b W,
//   ([h_0,h_0]) = ([h_2,h_2]) = sum a^2 H,  ([h_1,h_1]) = ([h_3,h_3]) = sum b^2 H,  ([h_0,h_1]) = ([h_2,h_3]) = sum a b H,
// and the products between a cos and a sin quadrature vanish (Re[R_nu conj R_mu] = 0).  fq[0..6] receive this SFT's terms of
// {Re sum a W, Im sum a W, Re sum b W, Im sum b W, sum a^2 H, sum b^2 H, sum a b H}, summed over the channels.
template <int CT, class CFG>
__device__ __forceinline__ void finish_terms(const KParams &p, const Tmpl &tm, const float2 *rt, const Track &tr, bool ok,
                                             float scale, float t, const float (&s1r)[CT], const float (&s1i)[CT],
                                             const float (&s2)[CT], const float (&us2)[CT], float &zr, float &zi, float &hh,
                                             float *fq = nullptr) {
  // |t| <= 1 + 1/2 + |b|/4: the MUFU sin/cos argument reduction (x/2pi rounded to fp32) stays below 3e-7 rad
  float sp, cp_;
  sincospi_fast(t, sp, cp_);
  const float as = scale * tr.amp;
  const float er = cp_ * as, ei = sp * as;
  const float a2 = as * tr.amp;
  const int resp = cfg_resp<CFG>(p);
  float sr = 0.f, si = 0.f, sh = 0.f;
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    // response (Eq.(5)-(6) P:80-85 as Lambda z = Re[R z]; DESIGN C3/D4)
    float2 R = tm.AE[c];
    if (fq) {                          // unit response; (a, b) are applied to the sums below
    } else if (resp == 1) {
      SFT_CHK_RANGE(p, rt + c * p.n_sft, 1, p.rtab, p.n_sl, CHK_RESP);
      const float2 r = __ldg(rt + c * p.n_sft);
      R = make_float2(tm.AE[c].x * r.x, tm.AE[c].x * r.y);      // AE is real here
    } else if (resp == 2) {
      SFT_CHK_RANGE(p, rt + c * p.n_sft, 1, p.rtab, p.n_sl, CHK_RESP);
      const float2 cs = __ldg(rt + c * p.n_sft);
      const float am = fmaf(p.depth, cs.x * tm.cl - cs.y * tm.sl, 1.0f);
      R = make_float2(R.x * am, R.y * am);
    }
    float gr, gi, r2;
    if (resp == 0 || fq) {             // AE is real
      gr = R.x * er; gi = R.x * ei; r2 = R.x * R.x;
    } else {
      gr = R.x * er - R.y * ei; gi = R.x * ei + R.y * er; r2 = R.x * R.x + R.y * R.y;   // p_c = R * A e^{i phi} pref
    }
    const float cr = gr * s1r[c] - gi * s1i[c], ci = gr * s1i[c] + gi * s1r[c];
    const float chh = r2 * a2 * us2[c] * s2[c];
    if (fq) {
      SFT_CHK_RANGE(p, rt + c * p.n_sft, 1, p.rtab, p.n_sl, CHK_RESP);
      const float2 ab = __ldg(rt + c * p.n_sft);
      const bool on = ok && us2[c] > 0.f;
      const float wa = on ? ab.x : 0.f, wb = on ? ab.y : 0.f, h_ = on ? chh : 0.f;
      const float xr = on ? cr : 0.f, xi_ = on ? ci : 0.f;
      if (c == 0) {
        fq[0] = wa * xr; fq[1] = wa * xi_; fq[2] = wb * xr; fq[3] = wb * xi_;
        fq[4] = wa * wa * h_; fq[5] = wb * wb * h_; fq[6] = wa * wb * h_;
      } else {
        fq[0] = fmaf(wa, xr, fq[0]); fq[1] = fmaf(wa, xi_, fq[1]); fq[2] = fmaf(wb, xr, fq[2]); fq[3] = fmaf(wb, xi_, fq[3]);
        fq[4] = fmaf(wa * wa, h_, fq[4]); fq[5] = fmaf(wb * wb, h_, fq[5]); fq[6] = fmaf(wa * wb, h_, fq[6]);
      }
    }
    if (CT == 1) {
      sr = cr; si = ci; sh = chh;
    } else {
      const bool present = us2[c] > 0.f;               // gaps hold zeros in the store, but guard 0 * garbage
      sr += present ? cr : 0.f;
      si += present ? ci : 0.f;
      sh += present ? chh : 0.f;
    }
  }
  zr = ok ? sr : 0.f;
  zi = ok ? si : 0.f;
  hh = ok ? sh : 0.f;
}

// Two consecutive SFTs (A = alpha, B = alpha + 1) of one template through the tier-1 moment tables at once: twice the
// independent work in one straight-line block (the fp64 tracks of alpha + 2 and alpha + 3 included), so that the
// fixed-latency dependency chains of one fill the issue gaps of the other.
template <int CT, class CFG>
__device__ __forceinline__ void duo_terms(const KParams &p, const Tmpl &tm, const float4 *Mrow0, int4 tb, const float2 *rt,
                                          const Track &trA, const Track &trB, bool goA, bool goB, const float (&usA)[CT],
                                          const float (&usB)[CT], double dnext, Track &nA, Track &nB, float &zrA, float &ziA,
                                          float &hhA, float &zrB, float &ziB, float &hhB) {
  const int j0A = trA.kc - p.kwin0, j0B = trB.kc - p.kwin0;
  const bool okA = goA && (unsigned)(j0A - 2) <= (unsigned)p.jmax, okB = goB && (unsigned)(j0B - 2) <= (unsigned)p.jmax;
  const bool fres = (cfg_kernel<CFG>(p) == 1);
  const float bA = fres ? trA.b : 0.f, bB = fres ? trB.b : 0.f;
  TableData<CT, 1> dA, dB;
  table_load<CT, 1>(p, fmaf(0.5f, bA, trA.x), bA, okA ? j0A - 2 : tb.y, tb.y, Mrow0, dA);
  table_load<CT, 1>(p, fmaf(0.5f, bB, trB.x), bB, okB ? j0B - 2 : tb.y, tb.y, Mrow0 + (unsigned)tb.w, dB);
  track_eval<CFG>(p, tm, dnext, nA);
  track_eval<CFG>(p, tm, dnext + 1.0, nB);
  float s1rA[CT], s1iA[CT], s2A[CT], s1rB[CT], s1iB[CT], s2B[CT];
  table_math2<CT, 1>(dA, dB, s1rA, s1iA, s2A, s1rB, s1iB, s2B);
  finish_terms<CT, CFG>(p, tm, rt, trA, okA, 1.0f, fmaf(2.0f, trA.frac, fmaf(0.25f, bA, trA.x)), s1rA, s1iA, s2A, usA, zrA, ziA, hhA);
  finish_terms<CT, CFG>(p, tm, rt + 1, trB, okB, 1.0f, fmaf(2.0f, trB.frac, fmaf(0.25f, bB, trB.x)), s1rB, s1iB, s2B, usB, zrB, ziB, hhB);
}

// Z_c = Re/Im of the per-(SFT, channel) complex term, H_c its <h,h> term (include/sft.h).
// Called by the whole warp as soon as one lane has an active pair (`go`); the other lanes run along on a
// clamped window and their results are discarded, so the control flow stays warp-uniform.
// `bmax` is the warp-wide max |b| of the active pairs: it selects the evaluator for the whole warp - the
// moment tables up to B_TABLE (if the plan has them), else the series order (a higher order than a lane
// needs is still correct for that lane) or the closed Fresnel form.  `Drow0` / `Mrow0` point at the row
// of SFT alpha, channel 0, in the pair-planar store / the moment table.  Also evaluates the track of the
// next SFT (see series_pairs).
template <int KT, int CT, class CFG>
__device__ __forceinline__ void pair_terms(const KParams &p, const Tmpl &tm, const float4 *Drow0, const float4 *Mrow0, int kb,
                                           float bt1, float bt2, const float2 *rt, const Track &tr, bool go, float bmax, const float (&us2)[CT],
                                           double dnext, Track &nxt, float &zr, float &zi, float &hh, float *fq = nullptr) {
  // window start in the zero-padded row; windows that miss the stored band entirely contribute 0
  const int j0 = tr.kc - p.kwin0;                                  // kwin0 = k_lo + K - PAD
  const bool ok = go && (unsigned)(j0 - 2) <= (unsigned)p.jmax;    // 2 <= j0 <= nb - 1 + PAD  <=>  window overlaps the band
  const int j0c = ok ? j0 : 2;
  const bool fres = (cfg_kernel<CFG>(p) == 1);
  const float b = fres ? tr.b : 0.f;
  float s1r[CT], s1i[CT], s2[CT];
  float scale;                 // the series evaluators return 2 pi J
  float t;                     // total phase / pi:  2 frac (= phi_a/pi) + prefactor phase / pi
  if (bmax <= bt2) {                   // bt1 / bt2: B_TABLE / B_TABLE2 where the warp's windows lie inside the block's table rows, else -1
    const float xp = fmaf(0.5f, b, tr.x);
    const int kci = ok ? j0 - 2 : kb;
    if (bmax <= bt1) table_eval<CT, CFG, 1>(p, tm, dnext, nxt, xp, b, kci, kb, Mrow0, s1r, s1i, s2);
    else table_eval<CT, CFG, 2>(p, tm, dnext, nxt, xp, b, kci, kb, Mrow0, s1r, s1i, s2);
    scale = 1.0f;
    t = fmaf(2.0f, tr.frac, fmaf(0.25f, b, tr.x));           // prefactor e^{i pi (x + b/4)}
  } else {
    Win w;
    win_init(p, Drow0, j0c, w);
    // the same window of the next SFT will be wanted next: pull its lines (both parity copies) into L1 now
    {
      const char *nE = (const char *)(w.dE + p.npair), *nO = (const char *)(w.dO + p.npair);
#pragma unroll
      for (int o = 0; o < (KT > 0 ? (KT + 1) * 16 + 127 : 128); o += 128) {
        asm volatile("prefetch.global.L1 [%0];" ::"l"(nE + o));
        asm volatile("prefetch.global.L1 [%0];" ::"l"(nO + o));
      }
    }
    Acc acc[CT];
#pragma unroll
    for (int c = 0; c < CT; ++c) {
      acc[c].A = make_float2(0.f, 0.f); acc[c].B = acc[c].A; acc[c].I = acc[c].A; acc[c].W = acc[c].A;
    }
    scale = INV_2PI_F;
    if (bmax <= B_ORDER3 || !(fabsf(b) > B_ORDER3)) {
      const float xp = fmaf(0.5f, b, tr.x);
      if (bmax == 0.f) series_pairs<0, KT, CT, CFG>(p, tm, dnext, nxt, xp, b, w, acc);
      else if (bmax <= B_ORDER1) series_pairs<1, KT, CT, CFG>(p, tm, dnext, nxt, xp, b, w, acc);
      else if (bmax <= B_ORDER2) series_pairs<2, KT, CT, CFG>(p, tm, dnext, nxt, xp, b, w, acc);
      else series_pairs<3, KT, CT, CFG>(p, tm, dnext, nxt, xp, b, w, acc);
      t = fmaf(2.0f, tr.frac, fmaf(0.25f, b, tr.x));         // prefactor e^{i pi (x + b/4)}
    } else {
      fresnel_pairs<KT, CT, CFG>(p, tm, dnext, nxt, tr.x, b, w, acc, scale);
      t = 2.0f * tr.frac;
    }
#pragma unroll
    for (int c = 0; c < CT; ++c) {
      s1r[c] = (acc[c].A.x + acc[c].A.y) - (acc[c].B.x + acc[c].B.y);
      s1i[c] = acc[c].I.x + acc[c].I.y;
      s2[c] = scale * (acc[c].W.x + acc[c].W.y);             // one of the two factors `scale` of |J|^2
    }
  }
  finish_terms<CT, CFG>(p, tm, rt, tr, ok, scale, t, s1r, s1i, s2, us2, zr, zi, hh, fq);
}

// ---------------------------------------------------------------------------------------------
// Fast path for "clean" blocks.  A block = up to SUB = 32 consecutive SFT slots of one work unit.
// It is clean when, for ALL 32 templates of the warp, every SFT of the block is active (DESIGN A12), its window lies
// in the stored band and |b| <= B_TABLE (tier-1 moment tables).  For an inspiral f, fdot, k_c and b grow with time and
// tau = t_c - t_a falls, so these conditions hold on the whole block iff they hold at its two end SFTs: they are
// decided ONCE per block (two closed-form track evaluations and one warp vote) instead of once per SFT, and the loop
// over the block's present SFTs then runs with no vote, no activity mask and no evaluator branch at all.
//
// Track inside a clean block.  With u = alpha - alpha_m (alpha_m = block start + 16) the closed forms of DESIGN W1 are
// powers of Theta = Theta_m (1 - eps u), eps = T / tau_m, so phase [cycles], y = f T (+ b/2) [bins], b and the amplitude
// are polynomials in u with geometrically falling coefficients:
//     phi/2pi (u) = sum_k p_k u^k,   p_k = -c_phase (-eps)^k [binom(5/8,k) Theta_m^(5/8) + c_phi binom(3/8,k) Theta_m^(3/8)],
//     f T   = d(phi/2pi)/du,    b = fdot T^2 = d(f T)/du        (exactly: dphi/dt = 2 pi f, t = alpha T),
// evaluated at degree 6 (phase) and 5 (y) - the terms up to u^2 by fp64 Horner, the small tail from u^3 on in fp32:
// 11 fp64 instructions per (template, SFT) instead of 33 - and by fp32 Horner at degree 2 / 3 for b / the amplitude.  The polynomial is used only where its first dropped term is
// below 5e-11 bins in y (so that k_c stays bit-identical to the closed form evaluated in fp64: a different k_c would
// need y within 5e-11 of a half-integer) and 1e-10 cycles in phase: |p_7| <= 5e-11 / (7 * 16^6); measured against
// 40-digit arithmetic the bound overestimates the actual error by ~1.2 (tests/test_gpu_parity.py checks k_c bit-exact).
// For config 2 that is tau_m >~ 9,000 s: 90 % of the SFTs.  Clean blocks closer to coalescence run the same loop with
// the closed-form fp64 track.
// ---------------------------------------------------------------------------------------------
constexpr int SUB = 32;                       // SFT slots per block of the fast path
// Validity of the polynomial track on a block (u in [-16, 15]); p_k = phase coefficients [cycles], y_k those of y [bins]:
constexpr double POLY_P7_MAX = 5e-11 / (7.0 * 16777216.0);      // phase after u^6, y after u^5: first dropped term 7 |p_7| 16^6 <= 5e-11 bins
constexpr double POLY_P5_MAX = 1e-7 / (20.0 * 4096.0);          // b after u^2: 20 |p_5| 16^3 <= 1e-7
constexpr double POLY_P3_MAX = 0.05 / 4096.0;                   // the terms from u^3 on are summed in fp32: |phase tail| <~ 0.05 cycles
constexpr double POLY_Y3_MAX = 5e-4 / 4096.0;                   //                                        |y tail| <~ 5e-4 bins
constexpr double POLY_EPS_MAX = 0.03 / 16.0;                    // amplitude after u^3: quartic term 0.08 (16 eps)^4 <= 7e-8

// u = j - 16 for slot j of a block: as double, and {u, u^3} as floats
static __constant__ double c_ud[SUB] = {-16., -15., -14., -13., -12., -11., -10., -9., -8., -7., -6., -5., -4., -3., -2., -1.,
                                 0.,   1.,   2.,   3.,   4.,   5.,   6.,   7.,  8.,  9.,  10., 11., 12., 13., 14., 15.};
static __constant__ float2 c_uf[SUB] = {{-16.f, -4096.f}, {-15.f, -3375.f}, {-14.f, -2744.f}, {-13.f, -2197.f}, {-12.f, -1728.f}, {-11.f, -1331.f},
                                 {-10.f, -1000.f}, {-9.f, -729.f},   {-8.f, -512.f},   {-7.f, -343.f},   {-6.f, -216.f},   {-5.f, -125.f},
                                 {-4.f, -64.f},    {-3.f, -27.f},    {-2.f, -8.f},     {-1.f, -1.f},     {0.f, 0.f},       {1.f, 1.f},
                                 {2.f, 8.f},       {3.f, 27.f},      {4.f, 64.f},      {5.f, 125.f},     {6.f, 216.f},     {7.f, 343.f},
                                 {8.f, 512.f},     {9.f, 729.f},     {10.f, 1000.f},   {11.f, 1331.f},   {12.f, 1728.f},   {13.f, 2197.f},
                                 {14.f, 2744.f},   {15.f, 3375.f}};

// Polynomial track of one template on one block.  The terms up to u^2 are kept in fp64 (the phase reaches 1e5+ cycles, y
// 1e2+ bins), the terms from u^3 on - below 0.05 cycles / 5e-4 bins by the validity test - are summed in fp32.
struct FastCoef {
  double p0, p1, p2;        // phase [cycles]
  double y0, y1, y2;        // y = f T + (Fresnel kernel: b/2) [bins]
  float pt[4];              // p_3 .. p_6
  float yt[3];              // y_3 .. y_5
  float bc[3];              // b = fdot T^2 (0 for the Dirichlet kernel)
  float ac[4];              // amplitude (f/F0)^(2/3) (x the template's amplitude constant where that is real)
};

// What the table evaluator needs of one (template, SFT).
struct FTrack {
  int kc;
  float xp;      // f T + b/2 - k_c  (b = 0 for the Dirichlet kernel)
  float b, frac, amp;
};

// Coefficients about slot 16 of the block starting at SFT g.  Returns false where the polynomial must not be used.
// `ascale` multiplies the amplitude polynomial.
template <class CFG>
__device__ __forceinline__ bool fast_coef(const KParams &p, const Tmpl &tm, int g, float ascale, FastCoef &fc) {
  const bool pn1 = cfg_pn1<CFG>(p) != 0, pn15 = cfg_pn1<CFG>(p) >= 2, fres = cfg_kernel<CFG>(p) == 1;
  const double tau = fma(-(double)(g + 16), p.T, tm.tau0);
  const double theta = tm.cTheta * tau;
  const float y0 = ex2_approx(-0.125f * lg2_approx((float)theta));
  const double y = (double)y0;
  const double y2 = y * y, y4 = y2 * y2, y8 = y4 * y4;
  const double r = fma(-theta, y8, 1.0);
  const double q = fma(y, fma(r, 9.0 / 128.0, 0.125) * r, y);       // Theta^(-1/8) (see track_eval_fp64)
  const double q2 = q * q, q3 = q2 * q, q4 = q2 * q2, q8 = q4 * q4;
  const double eps = (tm.cTheta * p.T) * q8;                         // T / tau_m
  const double me = -eps;
  double A = theta * q3;                                             // Theta^(5/8)
  double B = pn1 ? tm.cphi * (theta * (q3 * q2)) : 0.0;              // c_phi Theta^(3/8)
  double Cq = pn15 ? C15_PHI * (theta * (q3 * q3)) : 0.0;            // -3 pi/4 Theta^(1/4)
  const double mc = -tm.cphase;
  double pk[8];
  pk[0] = fma(mc, A + B + Cq, tm.phic_cyc);
#pragma unroll
  for (int k = 1; k <= 7; ++k) {
    A *= me * ((0.625 - (double)(k - 1)) / (double)k);               // binom(5/8, k) (-eps)^k Theta_m^(5/8)
    if (pn1) B *= me * ((0.375 - (double)(k - 1)) / (double)k);
    if (pn15) Cq *= me * ((0.25 - (double)(k - 1)) / (double)k);
    pk[k] = mc * (A + B + Cq);
  }
  double yk[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    const double ft = (double)(k + 1) * pk[k + 1];
    yk[k] = fres ? fma(0.5 * (double)((k + 1) * (k + 2)), pk[k + 2], ft) : ft;
  }
  fc.p0 = pk[0]; fc.p1 = pk[1]; fc.p2 = pk[2];
  fc.y0 = yk[0]; fc.y1 = yk[1]; fc.y2 = yk[2];
#pragma unroll
  for (int k = 0; k < 4; ++k) fc.pt[k] = (float)pk[3 + k];
#pragma unroll
  for (int k = 0; k < 3; ++k) fc.yt[k] = (float)yk[3 + k];
#pragma unroll
  for (int k = 0; k < 3; ++k) fc.bc[k] = fres ? (float)((double)((k + 1) * (k + 2)) * pk[k + 2]) : 0.f;
  // amplitude q^2 (1 + cf q^2)^(2/3) = a_m (1 - eps u)^(-s1),  s1 = -dln a/dln Theta = (1 + 2 w/3)/4,  w = cf q^2/(1 + cf q^2)
  double am = q2, s1 = 0.25;
  if (pn1) {
    const double gq = fma(tm.cf, q2, 1.0) + (pn15 ? C15_F * q3 : 0.0);
    am = q2 * (double)cbrtf((float)(gq * gq));                       // (1 + cf q^2 [+ c15 q^3])^(2/3) ~ 1.0x: fp32 cube root, 1e-7 relative
    s1 = 0.25 + (2.0 / 3.0) * (0.25 * tm.cf * q2 + (pn15 ? 0.375 * C15_F * q3 : 0.0)) / gq;
  }
  am *= (double)ascale;
  const double a1 = am * s1 * eps, a2 = a1 * (0.5 * (s1 + 1.0)) * eps, a3 = a2 * ((s1 + 2.0) * (1.0 / 3.0)) * eps;
  fc.ac[0] = (float)am; fc.ac[1] = (float)a1; fc.ac[2] = (float)a2; fc.ac[3] = (float)a3;
  return fabs(pk[7]) <= POLY_P7_MAX && fabs(pk[5]) <= POLY_P5_MAX && fabs(pk[3]) <= POLY_P3_MAX && fabs(yk[3]) <= POLY_Y3_MAX &&
         eps <= POLY_EPS_MAX && eps > 0.0;
}

// Kernel variants without CREG keep the coefficients in shared memory between the set-up of a block and its loop (26 registers
// per thread otherwise): 7 x 16 bytes per thread, laid out [vector][thread] so that every LDS.128 / STS.128 of a warp is conflict
// free.  Variants with CREG (compiled for 128 registers, 4 blocks per SM) keep them in registers: the loop of a clean block is
// bound by the L1 data pipe (ncu: l1tex__data_pipe_lsu_wavefronts 80 % of peak; a 128-bit load costs four wavefronts whatever its
// address pattern), and the 7 LDS.128 per two SFTs are a third of its wavefronts.
constexpr int COEF_V = 7;
__device__ __forceinline__ void coef_store(float4 *cs, const FastCoef &fc) {       // cs = slot of this thread
  *reinterpret_cast<double2 *>(cs) = make_double2(fc.p0, fc.p1);
  *reinterpret_cast<double2 *>(cs + TILE) = make_double2(fc.p2, fc.y0);
  *reinterpret_cast<double2 *>(cs + 2 * TILE) = make_double2(fc.y1, fc.y2);
  cs[3 * TILE] = make_float4(fc.pt[0], fc.pt[1], fc.pt[2], fc.pt[3]);
  cs[4 * TILE] = make_float4(fc.yt[0], fc.yt[1], fc.yt[2], fc.bc[0]);
  cs[5 * TILE] = make_float4(fc.bc[1], fc.bc[2], fc.ac[0], fc.ac[1]);
  cs[6 * TILE] = make_float4(fc.ac[2], fc.ac[3], 0.f, 0.f);
}

__device__ __forceinline__ void ftrack_poly1(const double2 d0, const double2 d1, const double2 d2, const float4 f3, const float4 f4,
                                             const float4 f5, const float2 f6, int j, FTrack &t) {
  const double u = c_ud[j];
  const float2 uu = c_uf[j];
  const float uf = uu.x;
  const float tp = uu.y * fmaf(fmaf(fmaf(f3.w, uf, f3.z), uf, f3.y), uf, f3.x);
  const float ty = uu.y * fmaf(fmaf(f4.z, uf, f4.y), uf, f4.x);
  const double ph = fma(fma(d1.x, u, d0.y), u, d0.x);
  const double yy = fma(fma(d2.y, u, d2.x), u, d1.y) + (double)ty;
  const double kr = yy + RND_MAGIC, pr = ph + RND_MAGIC;
  t.kc = __double2loint(kr);
  t.xp = (float)(yy - (kr - RND_MAGIC));
  t.frac = (float)(ph - (pr - RND_MAGIC)) + tp;
  t.b = fmaf(fmaf(f5.y, uf, f5.x), uf, f4.w);
  t.amp = fmaf(fmaf(fmaf(f6.y, uf, f6.x), uf, f5.w), uf, f5.z);
}

// tracks of slots jA and jB from the thread's coefficient slot
__device__ __forceinline__ void ftrack_poly2(const float4 *cs, int jA, int jB, FTrack &A, FTrack &B) {
  const double2 d0 = *reinterpret_cast<const double2 *>(cs);
  const double2 d1 = *reinterpret_cast<const double2 *>(cs + TILE);
  const double2 d2 = *reinterpret_cast<const double2 *>(cs + 2 * TILE);
  const float4 f3 = cs[3 * TILE], f4 = cs[4 * TILE], f5 = cs[5 * TILE];
  const float2 f6 = *reinterpret_cast<const float2 *>(cs + 6 * TILE);
  ftrack_poly1(d0, d1, d2, f3, f4, f5, f6, jA, A);
  ftrack_poly1(d0, d1, d2, f3, f4, f5, f6, jB, B);
}

// the same from coefficients held in registers (kernel variants with CREG)
__device__ __forceinline__ void ftrack_poly2r(const FastCoef &fc, int jA, int jB, FTrack &A, FTrack &B) {
  const double2 d0 = make_double2(fc.p0, fc.p1), d1 = make_double2(fc.p2, fc.y0), d2 = make_double2(fc.y1, fc.y2);
  const float4 f3 = make_float4(fc.pt[0], fc.pt[1], fc.pt[2], fc.pt[3]), f4 = make_float4(fc.yt[0], fc.yt[1], fc.yt[2], fc.bc[0]);
  const float4 f5 = make_float4(fc.bc[1], fc.bc[2], fc.ac[0], fc.ac[1]);
  const float2 f6 = make_float2(fc.ac[2], fc.ac[3]);
  ftrack_poly1(d0, d1, d2, f3, f4, f5, f6, jA, A);
  ftrack_poly1(d0, d1, d2, f3, f4, f5, f6, jB, B);
}

template <class CFG>
__device__ __forceinline__ void ftrack_closed(const KParams &p, const Tmpl &tm, double dalpha, float ascale, FTrack &t) {
  Track tr;
  track_eval_fp64<CFG>(p, tm, dalpha, tr);
  t.kc = tr.kc;
  t.b = (cfg_kernel<CFG>(p) == 1) ? tr.b : 0.f;
  t.xp = fmaf(0.5f, t.b, tr.x);
  t.frac = tr.frac;
  t.amp = tr.amp * ascale;
}

// Is the block [g, ge) clean for this warp (see above)?  Returns 0 = no (generic loop), 1 = clean, closed-form track,
// 2 = clean, polynomial track (coefficients in fc and, unless CREG, in the thread's shared-memory slot cs).  `mask` receives the
// block's presence bits (any channel), usv[c] the weight 1/s of SFT g + lane.
template <int CT, class CFG, bool CREG, bool BAND>
__device__ __forceinline__ int fast_setup(const KParams &p, const Tmpl &tm, int g, int ge, int lane, float ascale, float4 *cs,
                                          unsigned &mask, float (&usv)[CT], FastCoef &fc, int4 &tb) {
  bool pres = false;
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    SFT_CHK(p, g + lane >= ge || (unsigned long long)c * p.n_sft + g + lane < p.n_sl, CHK_US2);
    usv[c] = (g + lane < ge) ? __ldg(p.us2 + (size_t)c * p.n_sft + g + lane) : 0.f;
    pres |= usv[c] > 0.f;
  }
  mask = __ballot_sync(0xffffffffu, pres);
  if (mask == 0u || p.mtab == nullptr || cfg_phase<CFG>(p) != 0) return 0;
  if (BAND) {
    if ((g >> 5) != ((ge - 1) >> 5)) return 0;                     // (work units that are not aligned to the table's blocks of 32 SFTs)
    SFT_CHK(p, (unsigned long long)(g >> 5) < p.n_tblk, CHK_TBLK);
    tb = __ldg(p.tblk + (g >> 5));
    if (tb.z <= 0) return 0;
  } else {                                                         // full layout: row of SFT a at a * mrow0, all positions present
    tb = make_int4(0, 0, p.jmax + 1, 0);
  }
  const int kofs = p.kwin0 + 2 + tb.y;                              // window position of k_c inside the block's rows: k_c - kofs in [0, W)
  const bool fres = cfg_kernel<CFG>(p) == 1;
  const bool poly = __all_sync(0xffffffffu, fast_coef<CFG>(p, tm, g, ascale, fc));
  if (poly) {
    // the end SFTs from the polynomial itself (its error is far below the 1e-9 tie window of DESIGN A5/A12)
    auto end = [&](int j, double &fT, float &b, int &kc) {
      const double u = c_ud[j];
      const float2 uu = c_uf[j];
      const float ty = uu.y * fmaf(fmaf(fc.yt[2], uu.x, fc.yt[1]), uu.x, fc.yt[0]);
      const double yy = fma(fma(fc.y2, u, fc.y1), u, fc.y0) + (double)ty;
      b = fmaf(fmaf(fc.bc[2], uu.x, fc.bc[1]), uu.x, fc.bc[0]);
      kc = __double2loint(yy + RND_MAGIC);
      fT = fma(-0.5, (double)b, yy);                             // (b = 0 for the Dirichlet kernel: y = f T)
    };
    double fl, fh;
    float bl, bh;
    int kl, kh;
    end(0, fl, bl, kl);
    end(ge - 1 - g, fh, bh, kh);
    const double tau_h = fma(-(double)(ge - 1), p.T, tm.tau0);
    // Dirichlet kernel: the band edge test needs fdot T^2 although the evaluator does not (2 p_2 at the centre; +-1e-9 ties are flagged)
    const double b_edge = fres ? (double)bh : 2.0 * fc.p2;
    const bool ok = tau_h > p.T && fl >= p.f_loT && fh + b_edge <= p.f_hiT && (unsigned)(kl - kofs) < (unsigned)tb.z &&
                    (unsigned)(kh - kofs) < (unsigned)tb.z && bl >= 0.f && bh >= bl && bh <= p.b_table && kh >= kl;
    if (!__all_sync(0xffffffffu, ok)) return 0;
    if (!CREG) coef_store(cs, fc);
    return 2;
  }
  Track lo, hi;
  track_eval_fp64<CFG>(p, tm, (double)g, lo);
  track_eval_fp64<CFG>(p, tm, (double)(ge - 1), hi);
  const float bl = fres ? lo.b : 0.f, bh = fres ? hi.b : 0.f;
  const bool ok = lo.active && hi.active && (unsigned)(lo.kc - kofs) < (unsigned)tb.z && (unsigned)(hi.kc - kofs) < (unsigned)tb.z &&
                  bl >= 0.f && bh >= bl && bh <= p.b_table && hi.kc >= lo.kc;
  return __all_sync(0xffffffffu, ok) ? 1 : 0;
}

// table_load for a clean block: |xp| <= 1/2 (no clamp: the scale HTAB_R (1 - 2^-20) keeps xp = 1/2 inside the last cell), 32-bit
// table indices, no integer-to-float conversion.  `row` = float4 index of the SFT's row in mtab (channel 0).
template <int CT>
__device__ __forceinline__ void table_load_fast(const KParams &p, float xp, float b, int kcidx, unsigned row, TableData<CT, 1> &d) {
  constexpr float RM = 12582912.0f;
  const float cm = fmaf(xp, (float)HT1_R * (1.0f - 9.5367431640625e-7f), 0.5f * HT1_R - 0.5f) + RM;
  const unsigned cb = __float_as_uint(cm);
  const unsigned cellH = cb & (unsigned)(HT1_R - 1);
  const float cHf = cm - RM;                                                      // (float)cellH
  const float cSf = __uint_as_float(cb & ~(unsigned)((1 << HT1_SHIFT) - 1)) - RM;    // cell << HT1_SHIFT, cell = data-moment node
  const float4 *mp = p.mtab + (row + ((unsigned)kcidx * TAB_R + (cellH >> HT1_SHIFT)) * (unsigned)((TAB_Q + 1) / 2));
  const float4 *hp = p.htab1 + ((unsigned)kcidx * HT1_R + cellH);
#pragma unroll
  for (int c = 0; c < CT; ++c) {
    SFT_CHK_RANGE(p, mp + c * p.mchan, (TableData<CT, 1>::NL), p.mtab, p.n_mtab, CHK_MTAB_FAST);
    SFT_CHK_RANGE(p, hp + c * p.h1chan, 1, p.htab1, p.n_htab1, CHK_HTAB1_FAST);
#pragma unroll
    for (int i = 0; i < TableData<CT, 1>::NL; ++i) d.Mq[c][i] = __ldg(mp + c * p.mchan + i);
#pragma unroll
    for (int i = 0; i < TableData<CT, 1>::NHL; ++i) d.Hq[c][i] = __ldg(hp + c * p.h1chan + i);
  }
  d.aH = fmaf(cHf, -(2.0f * PI_F) / HT1_R, fmaf(xp, 2.0f * PI_F, (2.0f * PI_F) * (0.5f - 0.5f / HT1_R)));
  d.a = fmaf(cSf, -(2.0f * PI_F) / HT1_R, fmaf(xp, 2.0f * PI_F, (2.0f * PI_F) * (0.5f - 0.5f / TAB_R)));
  d.be = PI_F * b;
}

// Phase, amplitude, response and noise weight for a clean block (every lane active and in band).  Where the template's
// amplitude constant is real (no response) it is already inside `amp`.
template <int CT, class CFG>
__device__ __forceinline__ void finish_fast(const KParams &p, const Tmpl &tm, const float2 *rt, float amp, float t, const float (&s1r)[CT],
                                            const float (&s1i)[CT], const float (&s2)[CT], const float (&us2)[CT], float &zr, float &zi,
                                            float &hh) {
  if (CFG::RESP == 0 && CT == 1) {
    float sp, cp_;
    sincospi_fast(t, sp, cp_);
    const float er = cp_ * amp, ei = sp * amp;
    zr = er * s1r[0] - ei * s1i[0];
    zi = er * s1i[0] + ei * s1r[0];
    hh = (amp * amp) * (us2[0] * s2[0]);
  } else {
    Track tr;
    tr.amp = amp;
    finish_terms<CT, CFG>(p, tm, rt, tr, true, 1.0f, t, s1r, s1i, s2, us2, zr, zi, hh);
  }
}

// MODE 1, end of a work unit (32 SFT slots starting at g = 32 ch, n of them inside the data): the warp's tile holds the
// unit-local inclusive prefix sums (fp32, rows = lanes = templates), (axh, ahh) the unit's totals (fp64).  Single-pass scan
// with decoupled look-back along the SFT axis, one lane per template:
//   1. publish the unit's totals (aggregate) - nobody is waited for before this, so every claimed unit publishes;
//   2. walk back over the predecessors ch-1, ch-2, ... until one has published its INCLUSIVE totals (or the start is reached),
//      waiting where neither entry of a predecessor is there yet: units are claimed in ascending order from one counter, so
//      every predecessor is held by a resident warp that is past or on its way to step 1;
//   3. carry = inclusive(k) + aggregate(k+1) + ... + aggregate(ch-1), added in ASCENDING order: the same fp64 sums whichever
//      k the walk stopped at (run-to-run deterministic); publish carry + own totals as this unit's inclusive totals;
//   4. store carry + local prefix (carry split into hi + lo floats: <= 1 ulp of the fp32 output) transposed, as 128-byte rows
//      along the SFT axis, and snr = cum_xh / sqrt(cum_hh) (0 where cum_hh == 0).
// Records: a published entry is ONE 16-byte word {xh, hh} written and read by single 128-bit accesses, with the 16-bit
// epoch of the call in the low 8 mantissa bits of each double (2^-45 relative: invisible in the fp32 outputs).  A reader that
// finds the tag has the values, so no fence orders "data before flag" - a release fence here would wait for the 4 to 12 KB of
// output stores of the warp's previous unit to drain, 12 % of the kernel's stall samples when it was there.  Every sum is
// truncated to the 44-bit mantissa again (scan_trunc) so that a stored value equals the value its writer went on with.
__device__ __forceinline__ double scan_trunc(double v) {
  return __longlong_as_double(__double_as_longlong(v) & ~0xffll);
}
__device__ __forceinline__ void scan_publish(double2 *q, double xh, double hh, unsigned epoch) {      // xh, hh truncated
  const unsigned long long lo = (unsigned long long)__double_as_longlong(xh) | (epoch & 0xffu);
  const unsigned long long hi = (unsigned long long)__double_as_longlong(hh) | ((epoch >> 8) & 0xffu);
  asm volatile("{ .reg .b128 q; mov.b128 q, {%1, %2}; st.relaxed.gpu.global.b128 [%0], q; }" ::"l"(q), "l"(lo), "l"(hi) : "memory");
}
__device__ __forceinline__ bool scan_read(const double2 *q, unsigned epoch, double &xh, double &hh) {
  unsigned long long lo, hi;
  asm volatile("{ .reg .b128 q; ld.relaxed.gpu.global.b128 q, [%2]; mov.b128 {%0, %1}, q; }" : "=l"(lo), "=l"(hi) : "l"(q) : "memory");
  xh = __longlong_as_double((long long)(lo & ~0xffull));
  hh = __longlong_as_double((long long)(hi & ~0xffull));
  return (unsigned)((lo & 0xffu) | ((hi & 0xffu) << 8)) == epoch;
}
__device__ __forceinline__ void scan_store(const KParams &p, float *txh, float *thh, int tg, int ch, int n, int lane, long long t,
                                           double axh, double ahh, unsigned smask) {
  const bool ok = t < p.nT;
  const size_t nT = (size_t)p.nT;
  double cx = 0.0, chh = 0.0;
  if (ok) {
    const size_t me = (size_t)ch * nT + (size_t)t;
    SFT_CHK(p, me < p.n_scan, CHK_SCAN);
    axh = scan_trunc(axh);
    ahh = scan_trunc(ahh);
    scan_publish(p.scanA + me, axh, ahh, p.epoch);
    int k = ch - 1;
    double vx, vh;
    while (k >= 0) {
      const size_t e = (size_t)k * nT + (size_t)t;
      if (scan_read(p.scanP + e, p.epoch, vx, vh)) { cx = vx; chh = vh; break; }
      if (scan_read(p.scanA + e, p.epoch, vx, vh)) { --k; continue; }
      __nanosleep(64);
    }
    for (int j = k + 1; j < ch; ++j) {                  // (their tags were seen above: published, and written once per call)
      scan_read(p.scanA + (size_t)j * nT + (size_t)t, p.epoch, vx, vh);
      cx = scan_trunc(cx + vx); chh = scan_trunc(chh + vh);
    }
    scan_publish(p.scanP + me, scan_trunc(cx + axh), scan_trunc(chh + ahh), p.epoch);
  }
  // carry of row r (hi + lo floats) comes from lane r
  const float xhi = (float)cx, xlo = (float)(cx - (double)xhi), hhi = (float)chh, hlo = (float)(chh - (double)hhi);
  __syncwarp();
  const int g = ch * 32;
  // slot j shows the running sums of the last slot <= j that holds a value (smask); slots before the first one show 0:
  // slot 0 is made to hold that 0, so that every slot has a source
  if (!(smask & 1u)) {
    txh[lane * 33] = 0.f;
    thh[lane * 33] = 0.f;
    smask |= 1u;
    __syncwarp();
  }
  auto source = [&](int j) { return 31 - __clz(smask & (0xffffffffu >> (31 - j))); };
  const size_t al = (size_t)p.out_snr | (size_t)p.out_cx | (size_t)p.out_ch;   // (null = aligned)
  if ((p.n_sft & 3) == 0 && (al & 15) == 0) {
    // 4 rows x 32 slots per step: lane = (row r0 + lane / 8, slots 4 (lane % 8) ... + 3), 16-byte stores
    const int c4 = (lane & 7) * 4, rs = lane >> 3;
    int src[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) src[j] = source(c4 + j);
#pragma unroll 2
    for (int r0 = 0; r0 < 32; r0 += 4) {
      const int r = r0 + rs;
      const long long tt = (long long)tg * 32 + r;
      const float c0 = __shfl_sync(0xffffffffu, xhi, r), c1 = __shfl_sync(0xffffffffu, xlo, r);
      const float c2 = __shfl_sync(0xffffffffu, hhi, r), c3 = __shfl_sync(0xffffffffu, hlo, r);
      float x[4], h[4], q[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        x[j] = c0 + (c1 + txh[r * 33 + src[j]]);
        h[j] = c2 + (c3 + thh[r * 33 + src[j]]);
        q[j] = h[j] > 0.f ? x[j] * rsqrt_approx(h[j]) : 0.f;
      }
      if (tt < p.nT && c4 < n) {
        const size_t o = (size_t)tt * p.n_sft + g + c4;
        SFT_CHK(p, o + 4 <= p.n_out, CHK_OUT);
        if (p.out_snr) __stcs((float4 *)(p.out_snr + o), make_float4(q[0], q[1], q[2], q[3]));
        if (p.out_cx) __stcs((float4 *)(p.out_cx + o), make_float4(x[0], x[1], x[2], x[3]));
        if (p.out_ch) __stcs((float4 *)(p.out_ch + o), make_float4(h[0], h[1], h[2], h[3]));
      }
    }
  } else {
    const int sj = source(lane);
    for (int r = 0; r < 32; ++r) {
      const long long tt = (long long)tg * 32 + r;
      const float c0 = __shfl_sync(0xffffffffu, xhi, r), c1 = __shfl_sync(0xffffffffu, xlo, r);
      const float c2 = __shfl_sync(0xffffffffu, hhi, r), c3 = __shfl_sync(0xffffffffu, hlo, r);
      if (tt < p.nT && lane < n) {
        const float x = c0 + (c1 + txh[r * 33 + sj]);
        const float h = c2 + (c3 + thh[r * 33 + sj]);
        const size_t o = (size_t)tt * p.n_sft + g + lane;
        SFT_CHK(p, o < p.n_out, CHK_OUT);
        if (p.out_snr) __stcs(p.out_snr + o, h > 0.f ? x * rsqrt_approx(h) : 0.f);
        if (p.out_cx) __stcs(p.out_cx + o, x);
        if (p.out_ch) __stcs(p.out_ch + o, h);
      }
    }
  }
  __syncwarp();
}

// The loop over the present SFTs of a clean block, two at a time.  Accumulates into axh / ahh / axi (fp64; fp32 partial
// sums over the block).
template <int CT, int MODE, class CFG, bool POLY, bool CREG, bool BAND>
__device__ __forceinline__ void fast_block(const KParams &p, const Tmpl &tm, const float4 *cs, const FastCoef &fc, int4 tb, unsigned mask, const float (&usv)[CT],
                                           float ascale, int g, int ge, int tg, int lane, long long t, bool want_kc, double &axh,
                                           double &ahh, double &axi, float *txh, float *thh, unsigned long long *n_path) {
  const int n = ge - g;
  // first row of the block's table rows, shifted so that the GLOBAL window position indexes it (arithmetic mod 2^32)
  const unsigned mrow = BAND ? (unsigned)tb.w : p.mrow0;
  const unsigned row0 = BAND ? (unsigned)tb.x + (unsigned)(g & 31) * mrow - (unsigned)tb.y * (unsigned)(TAB_R * ((TAB_Q + 1) / 2))
                             : (unsigned)g * p.mrow0;
  const float2 *rt = p.rtab + g;
  int *kcp = (CFG::KC && want_kc) ? p.kc_out + ((size_t)(t < p.nT ? t : 0) * CT) * p.n_sft + g : nullptr;
  if (CFG::KC && kcp && t < p.nT) {
    for (int k = 0; k < n; ++k)
#pragma unroll
      for (int c = 0; c < CT; ++c) {
        SFT_CHK_RANGE(p, kcp + (size_t)c * p.n_sft + k, 1, p.kc_out, p.n_kc, CHK_KC);
        kcp[(size_t)c * p.n_sft + k] = -1;
      }
  }
  float fxh = 0.f, fhh = 0.f, fxi = 0.f;
  while (mask) {
    const int jA = __ffs(mask) - 1;
    mask &= mask - 1;
    const bool vB = mask != 0u;
    const int jB = vB ? __ffs(mask) - 1 : jA;
    mask &= mask - 1;                  // (0 stays 0)
    FTrack A, B;
    if (POLY) {
      if (CREG) ftrack_poly2r(fc, jA, jB, A, B);
      else ftrack_poly2(cs, jA, jB, A, B);
    } else {
      ftrack_closed<CFG>(p, tm, (double)(g + jA), ascale, A);
      ftrack_closed<CFG>(p, tm, (double)(g + jB), ascale, B);
    }
    float usA[CT], usB[CT];
#pragma unroll
    for (int c = 0; c < CT; ++c) {
      usA[c] = __shfl_sync(0xffffffffu, usv[c], jA);
      usB[c] = vB ? __shfl_sync(0xffffffffu, usv[c], jB) : 0.f;
    }
    TableData<CT, 1> dA, dB;
    table_load_fast<CT>(p, A.xp, A.b, A.kc - p.kwin0 - 2, row0 + (unsigned)jA * mrow, dA);
    table_load_fast<CT>(p, B.xp, B.b, B.kc - p.kwin0 - 2, row0 + (unsigned)jB * mrow, dB);
    float s1rA[CT], s1iA[CT], s2A[CT], s1rB[CT], s1iB[CT], s2B[CT];
    table_math2<CT, 1>(dA, dB, s1rA, s1iA, s2A, s1rB, s1iB, s2B);
    float zrA, ziA, hhA, zrB, ziB, hhB;
    // prefactor e^{i pi (x + b/4)},  x + b/4 = xp - b/4
    finish_fast<CT, CFG>(p, tm, rt + jA, A.amp, fmaf(2.0f, A.frac, fmaf(-0.25f, A.b, A.xp)), s1rA, s1iA, s2A, usA, zrA, ziA, hhA);
    finish_fast<CT, CFG>(p, tm, rt + jB, vB ? B.amp : 0.f, fmaf(2.0f, B.frac, fmaf(-0.25f, B.b, B.xp)), s1rB, s1iB, s2B, usB, zrB, ziB, hhB);
    if (CFG::KC && p.path_counts) {
      int np_ = 0;
#pragma unroll
      for (int c = 0; c < CT; ++c) np_ += (usA[c] > 0.f) + (vB && usB[c] > 0.f);
      n_path[PATH_TABLE] += (unsigned)__popc(__ballot_sync(0xffffffffu, t < p.nT)) * (unsigned)np_;
    }
    if (CFG::KC && kcp && t < p.nT) {
#pragma unroll
      for (int c = 0; c < CT; ++c) {
        SFT_CHK_RANGE(p, kcp + (size_t)c * p.n_sft + jA, 1, p.kc_out, p.n_kc, CHK_KC);
        SFT_CHK(p, !vB || (unsigned long long)(kcp + (size_t)c * p.n_sft + jB - p.kc_out) < p.n_kc, CHK_KC);
        if (usA[c] > 0.f) kcp[(size_t)c * p.n_sft + jA] = A.kc;
        if (vB && usB[c] > 0.f) kcp[(size_t)c * p.n_sft + jB] = B.kc;
      }
    }
    if (MODE == 1) {                   // running sums at the present slots only: scan_store fills the gaps.  fp32 inside the
      fxh += zrA; fhh += hhA;          // unit (<= 32 terms, as MODE 0 sums 8 SFTs in fp32); the carries across units are fp64
      txh[lane * 33 + jA] = fxh; thh[lane * 33 + jA] = fhh;
      if (vB) {
        fxh += zrB; fhh += hhB;
        txh[lane * 33 + jB] = fxh; thh[lane * 33 + jB] = fhh;
      }
    } else {
      fxh += zrA + zrB;
      fxi += ziA + ziB;
      fhh += hhA + hhB;
    }
  }
  if (MODE == 0) {
    axh += (double)fxh; axi += (double)fxi; ahh += (double)fhh;
  } else if (MODE == 1) {
    axh += (double)fxh; ahh += (double)fhh;      // (one block per unit: axh, ahh were 0)
  }
}

// ---------------------------------------------------------------------------------------------
// Main fused kernel.  Persistent grid; every warp draws (32 templates) x (SFT chunk) work units from
// p.counter.  CT == number of channels (exactly).
// MODE 0: chunk totals only (sft_reduce_kernel sums the chunks in fixed order).
// MODE 1 (cumulative): one work unit is one 32-SFT block; units are drawn in ascending SFT order, each
// publishes its aggregate and picks up the carry of all earlier units by decoupled look-back (scan_store),
// then writes the final cumulative <x,h>, <h,h> and SNR, transposed through shared memory so that global
// stores are 128-byte rows along the SFT axis.  One pass, no second kernel.
// MODE 2 (F-statistic): chunk totals of the seven sums of sft.h (sft_fstat).
// A work unit is walked in blocks of SUB = 32 SFT slots: clean blocks take the fast path above, all others the
// generic loop below, which runs in groups of GROUP SFTs: fp32 partial sums flushed into fp64 per group (MODE 0),
// one transposed store per group (MODE 1).
// ---------------------------------------------------------------------------------------------
template <int KT, int CT, int MODE, class CFG, int MINB, bool DUO, bool CREG, bool BAND = true>
__global__ void __launch_bounds__(TILE, MINB) sft_main_kernel(const KParams p) {
  constexpr int GROUP = MODE == 1 ? 32 : FLUSH;
  constexpr int TILE_F = 2 * 32 * 33;                  // two padded 32 x 32 tiles per warp
  __shared__ float tile_s[MODE == 1 ? (TILE / 32) * TILE_F : 1];
  __shared__ float4 coef_s[CREG ? 1 : COEF_V * TILE];  // polynomial-track coefficients of the current block, per thread
  float4 *cs = coef_s + (CREG ? 0 : threadIdx.x);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float *txh = tile_s + (MODE == 1 ? warp * TILE_F : 0);
  float *thh = txh + (MODE == 1 ? 32 * 33 : 0);
  const bool want_kc = CFG::KC && p.kc_out != nullptr;

  // Work units come from one counter.  A warp claims the unit AFTER the current one before it starts on the current one, so
  // that the latency of the atomic (3 % of the stall samples when it was waited for) hides under a unit's work: config 2
  // 0.2599 -> 0.2528 ms, config 3 1.2405 -> 1.2166 ms.  (MODE 1: the look-back of scan_store stays free of deadlock - a unit
  // waits only for units with smaller numbers, a warp's current unit has a smaller number than the one it holds in reserve,
  // so the smallest unpublished unit is always some warp's current unit, or the reserve of a warp that has already
  // published its current one.)  Single-channel variants only: the others sit at the register cap, and the extra live
  // register costs more in spills than the hidden latency returns (config 4, 2 channels: 0.4686 -> 0.4724 ms with it).
  // The first unit of every warp is its own number in the grid - no atomic: 2368 warps asking one address at the start of
  // the kernel cost ~5 us.
  constexpr bool PRECLAIM = CT == 1;
  int nxt = (int)blockIdx.x * (TILE / 32) + warp;
  bool first = true;
  for (;;) {
    int item = nxt;
    if (lane == 0) {
      if (PRECLAIM) nxt = p.first_dyn + atomicAdd(p.counter, 1);
      else if (!first) item = p.first_dyn + atomicAdd(p.counter, 1);
    }
    first = false;
    item = __shfl_sync(0xffffffffu, item, 0);
    if (item >= p.n_items) break;
    // MODE 0: latest (most expensive) chunks first; MODE 1: ascending, as the look-back of scan_store needs
    const int ch = MODE == 1 ? item / p.n_tgroups : p.n_chunks - 1 - item / p.n_tgroups;
    const int tg = item - (item / p.n_tgroups) * p.n_tgroups;
    const long long t = (long long)tg * 32 + lane;
    const int a0 = ch * p.chunk;
    const int a1 = min(a0 + p.chunk, p.n_sft);
    double afs[MODE == 2 ? 7 : 1];     // MODE 2: the seven sums of the F-statistic (finish_terms)
#pragma unroll
    for (int i = 0; i < (MODE == 2 ? 7 : 1); ++i) afs[i] = 0.0;
    double axh = 0.0, ahh = 0.0, axi = 0.0;
    unsigned long long n_path[PATH_N] = {0, 0, 0, 0, 0, 0, 0};
    unsigned smask = 0xffffffffu;      // MODE 1: slots of the unit's tile that were written (a clean block writes the present SFTs only)

    for (int gs = a0; gs < a1; gs += SUB) {
      const int gend = min(gs + SUB, a1);
      Tmpl tm;
      tmpl_load<CT>(p, t, tm);
      {
        unsigned mask;
        float usv[CT];
        // where the template's amplitude constant is real (no response, one channel) it is folded into the amplitude
        const float ascale = (CFG::RESP == 0 && CT == 1) ? tm.AE[0].x : 1.0f;
        FastCoef fc;
        int4 tbf;
        const int kind = MODE == 2 ? 0 : fast_setup<CT, CFG, CREG, BAND>(p, tm, gs, gend, lane, ascale, cs, mask, usv, fc, tbf);
        if (kind != 0) smask = mask;
        if (kind == 2) {
          fast_block<CT, MODE, CFG, true, CREG, BAND>(p, tm, cs, fc, tbf, mask, usv, ascale, gs, gend, tg, lane, t, want_kc, axh, ahh, axi, txh, thh, n_path);
          continue;
        }
        if (kind == 1) {
          fast_block<CT, MODE, CFG, false, CREG, BAND>(p, tm, cs, fc, tbf, mask, usv, ascale, gs, gend, tg, lane, t, want_kc, axh, ahh, axi, txh, thh, n_path);
          continue;
        }
      }
      // ---- generic loop over [gs, gend) ----
      double dalpha = (double)gs;
      const float *usp = p.us2 + gs;
      const float2 *rt = p.rtab + gs;
      const float4 *Drow0 = p.Dp + (size_t)gs * p.npair;
      int *kcp = want_kc ? p.kc_out + ((size_t)(t < p.nT ? t : 0) * CT) * p.n_sft + gs : nullptr;
      // table rows: one layout record per block of 32 SFT slots; [gs, gend) lies inside one block unless the work units are
      // not aligned to 32 (sft_plan_set_chunk), in which case the record is re-read per SFT
      const bool one_blk = (gs >> 5) == ((gend - 1) >> 5);
      int4 tb = !p.mtab ? make_int4(0, 0, 0, 0)
                : BAND  ? (SFT_CHK_TB(p, gs), __ldg(p.tblk + (gs >> 5)))
                        : make_int4((int)((unsigned)(gs & ~31) * p.mrow0), 0, p.jmax + 1, (int)p.mrow0);
      Track tr, tr2;                                   // tracks of SFT alpha and alpha + 1
      track_eval<CFG>(p, tm, dalpha, tr);
      track_eval<CFG>(p, tm, dalpha + 1.0, tr2);

      for (int g = gs; g < gend; g += GROUP) {
        const int ge = min(g + GROUP, gend);
        float fxh = 0.f, fhh = 0.f, fxi = 0.f;
        float ffs[MODE == 2 ? 7 : 1];
#pragma unroll
        for (int i = 0; i < (MODE == 2 ? 7 : 1); ++i) ffs[i] = 0.f;
        int alpha = g;
        while (alpha < ge) {
          float us2[CT], us2b[CT];
          bool any = false, anyb = false;
#pragma unroll
          for (int c = 0; c < CT; ++c) {
            SFT_CHK_RANGE(p, usp + c * p.n_sft, 1, p.us2, p.n_sl, CHK_US2);
            us2[c] = __ldg(usp + c * p.n_sft);
            any |= us2[c] > 0.f;                                   // warp-uniform
          }
          const bool go = any && tr.active && t < p.nT;
          const float ab = (go && cfg_kernel<CFG>(p) == 1) ? fabsf(tr.b) : 0.f;
          // the table rows of this SFT (block alpha >> 5) and whether the windows of all active lanes lie inside them
          if (!one_blk && p.mtab) {
            if (BAND) { SFT_CHK_TB(p, alpha); tb = __ldg(p.tblk + (alpha >> 5)); }
            else tb.x = (int)((unsigned)(alpha & ~31) * p.mrow0);
          }
          const float4 *Mrow0 = p.mtab + ((unsigned)tb.x + (unsigned)(alpha & 31) * (unsigned)tb.w);
          const int kci = tr.kc - p.kwin0 - 2;
          const bool tabok = !p.banded ? p.mtab != nullptr
                                       : (tb.z > 0 && __all_sync(0xffffffffu, !(go && (unsigned)kci <= (unsigned)p.jmax) ||
                                                                                  (unsigned)(kci - tb.y) < (unsigned)tb.z));
          const float bt1 = tabok ? p.b_table : -1.f, bt2 = tabok ? p.b_table2 : -1.f;
          // two SFTs at once when both are present and both go through the tier-1 tables
          bool duo = false, gob = false;
          if (DUO && MODE != 2 && alpha + 1 < ge && tabok && (alpha & 31) != 31) {
#pragma unroll
            for (int c = 0; c < CT; ++c) {
              SFT_CHK_RANGE(p, usp + c * p.n_sft + 1, 1, p.us2, p.n_sl, CHK_US2);
              us2b[c] = __ldg(usp + c * p.n_sft + 1);
              anyb |= us2b[c] > 0.f;
            }
            gob = anyb && tr2.active && t < p.nT;
            const float abb = (gob && cfg_kernel<CFG>(p) == 1) ? fabsf(tr2.b) : 0.f;
            const float bm2 = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(fmaxf(ab, abb))));
            const int kcb = tr2.kc - p.kwin0 - 2;
            const bool tabokb = !p.banded || __all_sync(0xffffffffu, !(gob && (unsigned)kcb <= (unsigned)p.jmax) || (unsigned)(kcb - tb.y) < (unsigned)tb.z);
            duo = tabokb && bm2 <= p.b_table && __any_sync(0xffffffffu, go) && __any_sync(0xffffffffu, gob);
          }
          if (duo) {
            Track nA, nB;
            float zrA, ziA, hhA, zrB, ziB, hhB;
            duo_terms<CT, CFG>(p, tm, Mrow0, tb, rt, tr, tr2, go, gob, us2, us2b, dalpha + 2.0, nA, nB, zrA, ziA, hhA, zrB, ziB, hhB);
            if (CFG::KC && p.path_counts) {
              int npa = 0, npb = 0;
#pragma unroll
              for (int c = 0; c < CT; ++c) { npa += us2[c] > 0.f; npb += us2b[c] > 0.f; }
              n_path[PATH_TABLE] += (unsigned)(__popc(__ballot_sync(0xffffffffu, go)) * npa + __popc(__ballot_sync(0xffffffffu, gob)) * npb);
            }
            if (CFG::KC && want_kc) {
              if (t < p.nT) {
#pragma unroll
                for (int c = 0; c < CT; ++c) {
                  SFT_CHK_RANGE(p, kcp + (size_t)c * p.n_sft, 2, p.kc_out, p.n_kc, CHK_KC);
                  kcp[(size_t)c * p.n_sft] = (tr.active && us2[c] > 0.f) ? tr.kc : -1;
                  kcp[(size_t)c * p.n_sft + 1] = (tr2.active && us2b[c] > 0.f) ? tr2.kc : -1;
                }
              }
              kcp += 2;
            }
            if (MODE == 1) {
              axh += (double)zrA; ahh += (double)hhA;
              txh[lane * 33 + (alpha - g)] = (float)axh;
              thh[lane * 33 + (alpha - g)] = (float)ahh;
              axh += (double)zrB; ahh += (double)hhB;
              txh[lane * 33 + (alpha + 1 - g)] = (float)axh;
              thh[lane * 33 + (alpha + 1 - g)] = (float)ahh;
            } else {
              fxh += zrA + zrB;
              fxi += ziA + ziB;
              fhh += hhA + hhB;
            }
            tr = nA; tr2 = nB;
            alpha += 2; dalpha += 2.0; usp += 2; rt += 2; Drow0 += 2 * p.npair;
            continue;
          }
          Track nxt;                                               // track of SFT alpha + 2
          if (__any_sync(0xffffffffu, go)) {
            const float bmax = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(ab)));
            if (CFG::KC && p.path_counts) {
              int n_present = 0;
#pragma unroll
              for (int c = 0; c < CT; ++c) n_present += us2[c] > 0.f;
              n_path[path_of(bmax, tabok)] += (unsigned)(__popc(__ballot_sync(0xffffffffu, go)) * n_present);
            }
            float zr, zi, hh;
            float fq[7];
            pair_terms<KT, CT, CFG>(p, tm, Drow0, Mrow0, tb.y, bt1, bt2, rt, tr, go, bmax, us2, dalpha + 2.0, nxt, zr, zi, hh, MODE == 2 ? fq : nullptr);
            if (MODE == 2) {
#pragma unroll
              for (int i = 0; i < 7; ++i) ffs[i] += fq[i];
            } else if (MODE == 1) {
              axh += (double)zr;
              ahh += (double)hh;
            } else {
              fxh += zr;
              fxi += zi;
              fhh += hh;
            }
          } else {
            track_eval<CFG>(p, tm, dalpha + 2.0, nxt);
          }
          if (CFG::KC && want_kc) {
            if (t < p.nT) {
#pragma unroll
              for (int c = 0; c < CT; ++c) {
                SFT_CHK_RANGE(p, kcp + (size_t)c * p.n_sft, 1, p.kc_out, p.n_kc, CHK_KC);
                kcp[(size_t)c * p.n_sft] = (tr.active && us2[c] > 0.f) ? tr.kc : -1;
              }
            }
            ++kcp;
          }
          tr = tr2;
          tr2 = nxt;
          if (MODE == 1) {
            txh[lane * 33 + (alpha - g)] = (float)axh;
            thh[lane * 33 + (alpha - g)] = (float)ahh;
          }
          ++alpha; dalpha += 1.0; ++usp; ++rt; Drow0 += p.npair;
        }
        if (MODE == 0) {
          axh += (double)fxh; axi += (double)fxi; ahh += (double)fhh;
        }
        if (MODE == 2) {
#pragma unroll
          for (int i = 0; i < 7; ++i) afs[i] += (double)ffs[i];
        }
      }
    }
    if (MODE == 1) {
      scan_store(p, txh, thh, tg, ch, a1 - a0, lane, t, axh, ahh, smask);        // (the host sets chunk = SUB = 32 for MODE 1)
    } else if (MODE == 2) {
      if (t < p.nT) {
        double *q = p.part + (size_t)ch * 7 * p.nT + t;
        SFT_CHK_RANGE(p, q + 6 * (size_t)p.nT, 1, p.part, p.n_part, CHK_PART);
#pragma unroll
        for (int i = 0; i < 7; ++i) q[(size_t)i * p.nT] = afs[i];
      }
    } else if (t < p.nT) {
      double *q = p.part + (size_t)ch * 3 * p.nT + t;
      SFT_CHK_RANGE(p, q + 2 * (size_t)p.nT, 1, p.part, p.n_part, CHK_PART);
      q[0] = axh;
      q[p.nT] = ahh;
      q[2 * p.nT] = axi;
    }
    if (CFG::KC && p.path_counts && lane == 0) {
#pragma unroll
      for (int i = 0; i < PATH_N; ++i)
        if (n_path[i]) atomicAdd(p.path_counts + i, n_path[i]);
    }
  }
}

#ifndef SFT_MAIN_ONLY
// Sum of the chunk totals in fp64, fixed order (deterministic).  grid = (ceil(nT/32), nq quantities),
// block = 32 templates x RED_SLICES chunk slices; slice s sums the chunks c = s (mod RED_SLICES).
constexpr int RED_SLICES = 16;
struct RedOut {
  double *q[7];          // output vector of quantity blockIdx.y (null: skipped)
};
__global__ void __launch_bounds__(32 * RED_SLICES) sft_reduce_kernel(const double *part, long long nT, int n_chunks, int nq, RedOut o) {
  __shared__ double sm[RED_SLICES][33];
  const int tx = threadIdx.x & 31, sl = threadIdx.x >> 5;
  const long long t = (long long)blockIdx.x * 32 + tx;
  double *out = o.q[blockIdx.y];
  if (!out) return;
  const size_t stride = (size_t)nq * nT;
  double s0 = 0.0, s1 = 0.0;
  if (t < nT) {
    const double *q = part + (size_t)blockIdx.y * nT + t;
    int c = sl;
    for (; c + RED_SLICES < n_chunks; c += 2 * RED_SLICES) {
      s0 += q[(size_t)c * stride];
      s1 += q[(size_t)(c + RED_SLICES) * stride];
    }
    if (c < n_chunks) s0 += q[(size_t)c * stride];
  }
  sm[sl][tx] = s0 + s1;
  __syncthreads();
  if (sl == 0 && t < nT) {
    double s = sm[0][tx];
#pragma unroll
    for (int j = 1; j < RED_SLICES; ++j) s += sm[j][tx];
    out[t] = s;
  }
}

// F-statistic from the seven sums (finish_terms): x = (Re Xa, Re Xb, Im Xa, Im Xb), M = [[A, C], [C, B]] (+) [[A, C], [C, B]],
//   2F = x^T M^-1 x = [B (x0^2 + x2^2) + A (x1^2 + x3^2) - 2 C (x0 x1 + x2 x3)] / (A B - C^2)            (Eq.(13))
// (0 where the determinant is not positive: no active SFT, or a and b proportional over the whole data).
__global__ void sft_fstat_kernel(long long n, const double *sums, double *twoF, double *xnu, double *mnu) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const double x0 = sums[t], x2 = sums[n + t], x1 = sums[2 * n + t], x3 = sums[3 * n + t];
  const double A = sums[4 * n + t], B = sums[5 * n + t], C = sums[6 * n + t];
  const double D = A * B - C * C;
  if (twoF) twoF[t] = D > 0.0 ? (B * (x0 * x0 + x2 * x2) + A * (x1 * x1 + x3 * x3) - 2.0 * C * (x0 * x1 + x2 * x3)) / D : 0.0;
  if (xnu) { xnu[t] = x0; xnu[n + t] = x1; xnu[2 * n + t] = x2; xnu[3 * n + t] = x3; }
  if (mnu) { mnu[t] = A; mnu[n + t] = B; mnu[2 * n + t] = C; }
}

// Validity of the per-SFT signal model, Eq.(33)-(34) P:244-248: the quadratic phase model Eq.(17) holds over
// one SFT while 1/2 T^2 max fddot <= delta df, i.e. delta_eff = 1/2 T^3 fddot <= delta.  fddot grows monotonically along an
// inspiral, so the largest value over a template's active SFTs (DESIGN A12) is the one of its LAST active SFT: the upper
// conditions (t_a + T < t_c, f_a + fdot_a T <= f_hi) hold up to some SFT index found by bisection, the lower one (f_lo <= f_a)
// from some index on.  One thread per template; pow() is fine here (once per template and bisection step).
__global__ void sft_validity_kernel(const KParams p, double delta_max, double *delta_eff, unsigned char *flags) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= p.nT) return;
  const double *row = p.params + t * 8;
  const double mc = row[0], eta = row[1], tau0 = row[2] - p.t0;
  const double M = mc * pow(eta, -0.6) * GMSUN_S;
  const double k = eta / (5.0 * M), F0 = 1.0 / (8.0 * 3.141592653589793 * M);
  const double cf = p.pn1 >= 1 ? (743.0 / 2688.0 + 11.0 / 32.0 * eta) : 0.0, c15 = p.pn1 >= 2 ? C15_F : 0.0;
  auto eval = [&](int a, double &fT, double &b, double &fdd) {
    const double tau = tau0 - (double)a * p.T;
    const double q = pow(k * tau, -0.125), q2 = q * q, q3 = q2 * q, q8 = q2 * q2 * q2 * q2;
    fT = F0 * p.T * q3 * (1.0 + cf * q2 + c15 * q3);
    b = F0 * k * p.T * p.T * (q8 * q3) * (0.375 + 0.625 * cf * q2 + 0.75 * c15 * q3);
    fdd = F0 * k * k * (q8 * q8 * q3) * (0.375 * 1.375 + 0.625 * 1.625 * cf * q2 + 0.75 * 1.75 * c15 * q3);
    return tau > p.T && fT + b <= p.f_hiT;                 // (NaN for tau <= 0 fails)
  };
  double fT, b, fdd, de = 0.0;
  if (eval(0, fT, b, fdd)) {
    int lo = 0, hi = p.n_sft - 1;                          // invariant: upper conditions hold at lo
    if (eval(hi, fT, b, fdd)) lo = hi;
    while (hi - lo > 1) {
      const int mid = lo + (hi - lo) / 2;
      if (eval(mid, fT, b, fdd)) lo = mid; else hi = mid;
    }
    eval(lo, fT, b, fdd);
    if (fT >= p.f_loT) de = 0.5 * p.T * p.T * p.T * fdd;
  }
  if (delta_eff) delta_eff[t] = de;
  if (flags) flags[t] = de > delta_max ? 1 : 0;
}

// Statistics on top of the inner products: log-likelihood L = <x,h> - <h,h>/2 (Eq.(2)) and the
// statistic maximised over distance and initial phase, (<x,h_c>^2 + <x,h_s>^2) / <h_c,h_c> (Eq.(7)-(9) P:97-101): shifting
// phi_c by pi/2 turns the complex sum Z into iZ, so <x,h_c> = Re Z = xh, <x,h_s> = -Im Z, and <h_c,h_c> = <h_s,h_s> = hh.
__global__ void sft_statistics_kernel(long long n, const double *xh, const double *xi, const double *hh, double *loglike,
                                      double *rho2max) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const double a = xh[t], b = xi[t], h = hh[t];
  if (loglike) loglike[t] = a - 0.5 * h;
  if (rho2max) rho2max[t] = h > 0.0 ? (a * a + b * b) / h : 0.0;
}

// Whitening of one channel at load time (Eq.(15); DESIGN "store"): writes both pair-planar
// copies of the zero-padded row of SFT a.  Padded index j <-> bin k = k_lo + j - PAD.
__global__ void sft_whiten_kernel(const float2 *raw, const double *psd_scale, const double *psd_shape, int n_sft,
                                  int nb, int k_lo, int kv_lo, int kv_hi, int PAD, int npair, double T, double S_ref,
                                  float4 *Dp0, float4 *Dp1, float *us2) {
  const int a = blockIdx.x;
  const double s = psd_scale[a];
  const bool present = isfinite(s) && s > 0.0;
  if (threadIdx.x == 0) us2[a] = present ? (float)(1.0 / s) : 0.f;
  const double pre = present ? 2.0 * sqrt(S_ref / T) / s : 0.0;
  auto value = [&](int j) {
    const int jj = j - PAD, k = k_lo + jj;
    float2 o = make_float2(0.f, 0.f);
    if (present && jj >= 0 && jj < nb && k >= kv_lo && k < kv_hi) {
      const double Sk = psd_shape ? psd_shape[jj] : 1.0;
      const float2 v = raw[(size_t)a * nb + jj];
      const double w = pre / Sk;
      o = make_float2((float)(w * (double)v.x), (float)(-w * (double)v.y));
    }
    return o;
  };
  for (int i = threadIdx.x; i < 2 * npair; i += blockDim.x) {
    const int copy = i >= npair, e = copy ? i - npair : i;
    const float2 lo = value(2 * e + copy), hi = value(2 * e + copy + 1);
    (copy ? Dp1 : Dp0)[(size_t)a * npair + e] = make_float4(lo.x, hi.x, lo.y, hi.y);
  }
}

__global__ void sft_ub2_kernel(const double *psd_shape, int nb, int k_lo, int kv_lo, int kv_hi, int PAD, int npair,
                               double S_ref, float2 *ub0, float2 *ub1) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 2 * npair) return;
  const int copy = i >= npair, e = copy ? i - npair : i;
  auto value = [&](int j) {
    const int jj = j - PAD, k = k_lo + jj;
    if (jj < 0 || jj >= nb || k < kv_lo || k >= kv_hi) return 0.f;
    return (float)(S_ref / (psd_shape ? psd_shape[jj] : 1.0));
  };
  (copy ? ub1 : ub0)[e] = make_float2(value(2 * e + copy), value(2 * e + copy + 1));
}

// SFT_RESP_ANNUAL: (cos, sin)(2 pi t_a / P + psi_c) per (channel, SFT).
__global__ void sft_annual_table_kernel(int n_sft, double t0, double T, double period, double psi, float2 *out) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= n_sft) return;
  double s, c;
  sincos(2.0 * 3.141592653589793 * ((t0 + (double)a * T) / period) + psi, &s, &c);
  out[a] = make_float2((float)c, (float)s);
}

#endif  // SFT_MAIN_ONLY

}  // namespace sftk
