// psfft_f32_fft.cu -- float instantiations of the launchers, group FFT (psfft_launch_impl.cuh).
#include "psfft_launch_impl.cuh"
namespace psfft {
PSFFT_INSTANTIATE_FFT(float)
}
