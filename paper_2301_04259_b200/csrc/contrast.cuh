// SOAPcontrast: "each wavelength pixel is first accessed by the global index of the kernel.  Next on each
// thread, it derives the contrast by calculating the ratio of two Planck functions at two different effective
// temperatures."  The wavelength-dependent I_ratio of Eq. 3 for a spot or facula modelled by a temperature:
//     contrast[m] = B_lambda(T_active) / B_lambda(T_quiet) = expm1(h c / (lambda_m k_B T_quiet)) / expm1(h c / (lambda_m k_B T_active)),
// lambda_m = lambda0 + m dlambda in Angstrom.  (SOAP 2.0 used the single value at 5293 A.)
// One thread per pixel, evaluated in fp64 and rounded once to the output type: 310 000 pixels are launch-latency sized,
// not a cost centre.
#pragma once
#include <cuda_runtime.h>

namespace soap {

// h c / k_B in Angstrom Kelvin from the exact SI values of the 2019 redefinition:
// 6.62607015e-34 J s * 299792458 m/s / 1.380649e-23 J/K = 1.4387768775...e-2 m K
constexpr double kSecondRadiationConstantAngstromK = 6.62607015e-34 * 299792458.0 / 1.380649e-23 * 1e10;

template <typename T>
__global__ void __launch_bounds__(256) contrast_planck_kernel(double lambda0, double dlambda, long long n_pix, double inv_t_quiet,
                                                              double inv_t_active, T *__restrict__ out) {
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n_pix) return;
    const double c2_over_lambda = kSecondRadiationConstantAngstromK / (lambda0 + dlambda * (double)m);
    out[m] = (T)(expm1(c2_over_lambda * inv_t_quiet) / expm1(c2_over_lambda * inv_t_active));
}

}  // namespace soap
