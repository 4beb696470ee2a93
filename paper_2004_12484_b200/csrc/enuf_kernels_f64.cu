// All kernels of the ENUF path instantiated for T = double.
#include "enuf_launch.cuh"

namespace enuf {
template int configure_kernels<double>(enuf_plan*);
template int spread_ctas_per_sm<double>(int);
template int launch_bin<double>(enuf_plan*, const void*, const void*, void*);
template int launch_spread<double>(enuf_plan*);
template int launch_fft<double>(enuf_plan*);
template int launch_fft_forward<double>(enuf_plan*);
template int launch_fft_backward<double>(enuf_plan*);
template int launch_gather<double>(enuf_plan*, void*);
template int launch_real<double>(enuf_plan*, const void*, const void*, double, int, void*);
}  // namespace enuf
