// sft_var_lisa.cu - main-kernel variants of the LISA configuration (4): two channels, annual response, K = 16; and the
// F-statistic sums (MODE 2, run-time flags, one or two channels).
#define SFT_MAIN_ONLY
#include "sft_launch.cuh"

namespace sftl {

template <int MODE>
static bool go(const Key &key, const Ctx &c, const sftk::KParams &k) {
  if (key.lisa && key.C == 2 && key.K == 16) { launch_variant<16, 2, MODE, CfgLISA, true>(c, k); return true; }
  return false;
}

bool launch_lisa(const Key &key, const Ctx &c, const sftk::KParams &k) {
  if (key.mode == 0) return go<0>(key, c, k);
  if (key.mode == 1) return go<1>(key, c, k);
  if (key.mode == 2 && key.C == 1) { launch_variant<0, 1, 2, CfgAny>(c, k); return true; }
  if (key.mode == 2 && key.C == 2) { launch_variant<0, 2, 2, CfgAny>(c, k); return true; }
  return false;
}

}  // namespace sftl
