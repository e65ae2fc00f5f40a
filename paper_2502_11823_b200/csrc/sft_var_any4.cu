// sft_var_any4.cu - main-kernel variant with run-time flags (any kernel / PN order / response / phase path; k_c output and
// evaluator-path counters) for 4 channel(s).
#define SFT_MAIN_ONLY
#include "sft_launch.cuh"

namespace sftl {

bool launch_any4(const Key &key, const Ctx &c, const sftk::KParams &k) {
  if (key.C != 4 && !(4 == 4 && key.C > 4)) return false;
  if (key.mode == 0) { launch_variant<0, 4, 0, CfgAny>(c, k); return true; }
  if (key.mode == 1) { launch_variant<0, 4, 1, CfgAny>(c, k); return true; }
  return false;
}

}  // namespace sftl
