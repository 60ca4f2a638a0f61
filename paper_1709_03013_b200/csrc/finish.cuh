// Finishing step: counts -> S, one CTA (csrc/csg.cu: finish_action_kernel; also the tail of the fused small-N launch
// of bitset_action_kernel).
//   eps == 1, dim 2: Eq. 4 with n_i = counts[i-1]:  S = 2 (N - 2 N_0 + 4 N_1 - 2 N_2)
//   eps == 1, dim 4: S = (4/sqrt 6)(N - N_0 + 9 N_1 - 16 N_2 + 8 N_3)   (not in the paper; A8)
//   eps <  1, dim 2: Eq. 5: S = 2 eps [N - 2 eps sum_k N_k f_2(k, eps)],
//                    f_2(k,e) = (1-e)^k - 2 e k (1-e)^(k-1) + e^2 k(k-1)/2 (1-e)^(k-2)   (bracket multiplied out)
//   eps <  1, dim 4: S = (4/sqrt 6) sqrt(eps) [N - eps sum_k N_k f_4(k, eps)]   (not in the paper; A9),
//                    f_4(k,e) = (1-e)^k - 9 e k (1-e)^(k-1) + 8 e^2 k(k-1) (1-e)^(k-2) - (4/3) e^3 k(k-1)(k-2) (1-e)^(k-3)
// The integer combinations are exact in int64 and below 2^53, so the local S is one exact product.
// The smeared sum is a fixed-order double reduction: FIN_LANES virtual lanes, lane l sums the bins k = l (mod FIN_LANES)
// in ascending order with Kahan compensation, then a binary tree over the lanes.  The order does not depend on how many
// threads walk the lanes, so every launch shape gives the same bits.
#pragma once

namespace csg {

constexpr int FIN_LANES = 1024;

// Whole CTA must call it (blockDim.x divides FIN_LANES); red: FIN_LANES doubles of shared memory.
__device__ __forceinline__ void finish_block(const long long* __restrict__ counts, long long N, int dim, double eps,
                                             int kmax, double* __restrict__ S, double* red) {
    const int tid = threadIdx.x, nthr = blockDim.x;
    if (eps == 1.0) {
        if (tid == 0) {
            if (dim == 2) {
                const long long I2 = N - 2 * counts[0] + 4 * counts[1] - 2 * counts[2];
                *S = 2.0 * (double)I2;
            } else {
                const long long I4 = N - counts[0] + 9 * counts[1] - 16 * counts[2] + 8 * counts[3];
                *S = (4.0 / sqrt(6.0)) * (double)I4;
            }
        }
        return;
    }
    const double x = 1.0 - eps;
    for (int l = tid; l < FIN_LANES; l += nthr) {
        double sum = 0.0, comp = 0.0;
        for (long long k = l; k <= kmax; k += FIN_LANES) {
            const long long c = counts[k];
            if (c == 0) continue;
            const double dk = (double)k;
            double w = pow(x, dk);
            if (dim == 2) {
                if (k >= 1) w -= 2.0 * eps * dk * pow(x, dk - 1.0);
                if (k >= 2) w += 0.5 * eps * eps * dk * (dk - 1.0) * pow(x, dk - 2.0);
            } else {
                if (k >= 1) w -= 9.0 * eps * dk * pow(x, dk - 1.0);
                if (k >= 2) w += 8.0 * eps * eps * dk * (dk - 1.0) * pow(x, dk - 2.0);
                if (k >= 3) w -= (4.0 / 3.0) * eps * eps * eps * dk * (dk - 1.0) * (dk - 2.0) * pow(x, dk - 3.0);
            }
            const double term = (double)c * w;
            const double y = term - comp;
            const double t = sum + y;
            comp = (t - sum) - y;
            sum = t;
        }
        red[l] = sum;
    }
    __syncthreads();
    for (int s = FIN_LANES / 2; s > 0; s >>= 1) {
        for (int l = tid; l < s; l += nthr) red[l] += red[l + s];
        __syncthreads();
    }
    if (tid == 0) {
        if (dim == 2) *S = 2.0 * eps * ((double)N - 2.0 * eps * red[0]);
        else *S = (4.0 / sqrt(6.0)) * sqrt(eps) * ((double)N - eps * red[0]);
    }
}

}  // namespace csg
