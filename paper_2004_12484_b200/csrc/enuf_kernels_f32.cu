// All kernels of the ENUF path instantiated for T = float.
#include "enuf_launch.cuh"

namespace enuf {
template int configure_kernels<float>(enuf_plan*);
template int spread_ctas_per_sm<float>(int);
template int launch_bin<float>(enuf_plan*, const void*, const void*, void*);
template int launch_spread<float>(enuf_plan*);
template int launch_fft<float>(enuf_plan*);
template int launch_fft_forward<float>(enuf_plan*);
template int launch_fft_backward<float>(enuf_plan*);
template int launch_gather<float>(enuf_plan*, void*);
template int launch_real<float>(enuf_plan*, const void*, const void*, double, int, void*);
}  // namespace enuf
