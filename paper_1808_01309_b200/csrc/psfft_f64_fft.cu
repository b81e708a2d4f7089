// psfft_f64_fft.cu -- double instantiations of the launchers, group FFT (psfft_launch_impl.cuh).
#include "psfft_launch_impl.cuh"
namespace psfft {
PSFFT_INSTANTIATE_FFT(double)
}
