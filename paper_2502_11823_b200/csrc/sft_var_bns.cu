// sft_var_bns.cu - main-kernel variants of the ET-BNS configurations (2, 3, 5): K = 8, one channel, no response.
#define SFT_MAIN_ONLY
#include "sft_launch.cuh"

namespace sftl {

template <int MODE>
static bool go(const Key &key, const Ctx &c, const sftk::KParams &k) {
  if (key.bns32) { launch_variant<8, 1, MODE, CfgBNS32>(c, k); return true; }
  if (key.bns && key.C == 1 && key.K == 8) { launch_variant<8, 1, MODE, CfgBNS, true>(c, k); return true; }
  return false;
}

bool launch_bns(const Key &key, const Ctx &c, const sftk::KParams &k) {
  if (key.mode == 0) return go<0>(key, c, k);
  if (key.mode == 1) return go<1>(key, c, k);
  return false;
}

}  // namespace sftl
