// cdh_rdf.cuh -- g(r) from a summed histogram (Eqs. 1-3).
//   p_kappa = hist[kappa] / N_frames;  g_kappa = p_kappa / (4 pi (N_pairs / V) r^2 dr),  dr = r_max / n_bins,
//   r = (kappa + 1/2) dr (reading Q15).  Plain IEEE double operations in the order of the formula, one
// thread per bin: O(n_hist * n_bins), HBM-bound and negligible next to the histogram itself.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cdh {

struct RdfParams {
    const unsigned long long* hist;   // [n_hist][n_bins]
    const double* density;            // [n_hist]  N_pairs / V (one rounded division on the host)
    double* g;                        // [n_hist][n_bins]
    double dr, n_frames;
    uint32_t n_bins;
    uint64_t total;                   // n_hist * n_bins
};

__global__ void __launch_bounds__(256) rdf_kernel(const RdfParams P) {
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= P.total) return;
    const uint32_t h = (uint32_t)(t / P.n_bins), k = (uint32_t)(t % P.n_bins);
    const double four_pi = __dmul_rn(4.0, 3.14159265358979323846);
    const double r = __dmul_rn(__dadd_rn((double)k, 0.5), P.dr);
    const double shell = __dmul_rn(__dmul_rn(four_pi, __dmul_rn(r, r)), P.dr);
    const double p = __ddiv_rn(__ull2double_rn(P.hist[t]), P.n_frames);
    P.g[t] = __ddiv_rn(p, __dmul_rn(__ldg(P.density + h), shell));
}

}  // namespace cdh
