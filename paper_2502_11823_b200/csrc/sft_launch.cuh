// sft_launch.cuh - launch of the fused main kernel (sft_kernels.cuh :: sft_main_kernel).  Its template variants are
// instantiated in several translation units (sft_var_*.cu) that compile in parallel; sft_lib.cu asks them in turn.
#pragma once
#include <cuda_runtime.h>
#include "sft_kernels.cuh"

#ifndef SFT_DUO
#define SFT_DUO true        // two consecutive SFTs per step through the tier-1 tables (sft_kernels.cuh :: duo_terms)
#endif
#ifndef SFT_CREG_MINB
#define SFT_CREG_MINB 4     // resident blocks per SM of the CREG variants (128 registers)
#endif
#ifndef SFT_MINB
#define SFT_MINB 5          // resident 128-thread blocks per SM the other variants are compiled for
#endif

namespace sftl {

// Compile-time flag sets of the hot variants (everything else takes the run-time-flag variant):
//   CfgBNS  = Fresnel kernel, 0PN+1PN, no response      (configs 2, 3, 5)
//   CfgNewt = Fresnel kernel, 0PN, no response          (config 1)
//   CfgLISA = Fresnel kernel, 0PN+1PN, annual response  (config 4)
//   CfgAny  = run-time flags (incl. the phase path), optional k_c output and path counters
using CfgBNS = sftk::Cfg<1, 1, 0, 0>;
using CfgNewt = sftk::Cfg<1, 0, 0, 0>;
using CfgLISA = sftk::Cfg<1, 1, 2, 0>;
using CfgAny = sftk::Cfg<-1, -1, -1, 1, -1>;
using CfgBNS32 = sftk::Cfg<1, 1, 0, 0, 1>;    // CfgBNS with the split-fp32 (double-float) phase track (config 5)

struct Ctx {
  cudaStream_t stream;
  int n_sm;
  bool banded;             // the plan's moment tables follow a track (sft_plan_set_table_track)
};

// What a call needs of the kernel: MODE 0 totals, 1 cumulative, 2 F-statistic sums; which flag set fits.
struct Key {
  int mode, C, K;
  bool bns32, bns, newt, lisa;
};

// CREG: polynomial-track coefficients in registers (128 registers, 4 blocks per SM) instead of shared memory (96, 5 blocks).
// BAND = false: specialisation for the full table layout: row addresses from a constant-bank operand (only CREG variants have it).
template <int KT, int CT, int MODE, class CFG, bool CREG = false, bool BAND = true>
static void launch_variant(const Ctx &c, const sftk::KParams &k) {
  if (CREG && BAND && !c.banded) return launch_variant<KT, CT, MODE, CFG, CREG, false>(c, k);
  auto kern = sftk::sft_main_kernel<KT, CT, MODE, CFG, CREG ? SFT_CREG_MINB : SFT_MINB, SFT_DUO, CREG, BAND>;
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, sftk::TILE, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
  long long blocks = (long long)c.n_sm * per_sm;
  const long long need = ((long long)k.n_items + sftk::TILE / 32 - 1) / (sftk::TILE / 32);
  if (blocks > need) blocks = need;
  sftk::KParams kk = k;
  kk.first_dyn = (int)blocks * (sftk::TILE / 32);      // units 0 .. first_dyn - 1 belong to the grid's warps, the rest to the counter
  kern<<<(unsigned)blocks, sftk::TILE, 0, c.stream>>>(kk);
}

// One per translation unit: launches and returns true if the unit holds the variant for `key`.
bool launch_bns(const Key &key, const Ctx &c, const sftk::KParams &k);     // sft_var_bns.cu:  config-2/3/5 variants (K = 8)
bool launch_misc(const Key &key, const Ctx &c, const sftk::KParams &k);    // sft_var_misc.cu: other BNS widths, Newtonian K = 4
bool launch_lisa(const Key &key, const Ctx &c, const sftk::KParams &k);    // sft_var_lisa.cu: config 4; F-statistic sums
bool launch_any1(const Key &key, const Ctx &c, const sftk::KParams &k);    // sft_var_any1..4.cu: run-time flags, 1..4 channels
bool launch_any2(const Key &key, const Ctx &c, const sftk::KParams &k);
bool launch_any3(const Key &key, const Ctx &c, const sftk::KParams &k);
bool launch_any4(const Key &key, const Ctx &c, const sftk::KParams &k);

}  // namespace sftl
