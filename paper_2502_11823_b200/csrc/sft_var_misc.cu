// sft_var_misc.cu - main-kernel variants with compile-time flags for other band widths of the BNS recipe (config 5's K axis)
// and for the Newtonian chirp of config 1.
#define SFT_MAIN_ONLY
#include "sft_launch.cuh"

namespace sftl {

template <int MODE>
static bool go(const Key &key, const Ctx &c, const sftk::KParams &k) {
  if (key.bns && key.C == 1 && key.K == 16) { launch_variant<16, 1, MODE, CfgBNS>(c, k); return true; }
  if (key.bns && key.C == 1) { launch_variant<0, 1, MODE, CfgBNS>(c, k); return true; }
  if (key.newt && key.C == 1 && key.K == 4) { launch_variant<4, 1, MODE, CfgNewt>(c, k); return true; }
  return false;
}

bool launch_misc(const Key &key, const Ctx &c, const sftk::KParams &k) {
  if (key.mode == 0) return go<0>(key, c, k);
  if (key.mode == 1) return go<1>(key, c, k);
  return false;
}

}  // namespace sftl
