// sft_var_any1.cu - main-kernel variant with run-time flags (any kernel / PN order / response / phase path; k_c output and
// evaluator-path counters) for 1 channel(s).
#define SFT_MAIN_ONLY
#include "sft_launch.cuh"

namespace sftl {

bool launch_any1(const Key &key, const Ctx &c, const sftk::KParams &k) {
  if (key.C != 1 && !(1 == 4 && key.C > 4)) return false;
  if (key.mode == 0) { launch_variant<0, 1, 0, CfgAny>(c, k); return true; }
  if (key.mode == 1) { launch_variant<0, 1, 1, CfgAny>(c, k); return true; }
  return false;
}

}  // namespace sftl
