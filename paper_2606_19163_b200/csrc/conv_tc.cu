// conv_tc.cu - tcgen05 / TMEM / TMA implicit-GEMM convolutions (placeholder until the
// tensor-core kernels land: reports "unsupported" so the executor uses conv_simt).
#include "kernels.h"
namespace pulse {
bool conv_tc_supported(const ConvArgs&) { return false; }
int conv_tc(const ConvArgs&, cudaStream_t) { return 0; }
bool wgrad_tc_supported(const WgradArgs&) { return false; }
int wgrad_tc(const WgradArgs&, cudaStream_t) { return 0; }
const char* tc_last_error() { return ""; }
}  // namespace pulse
