// taylor.cuh -- index helpers and the Taylor shift of an order-3 local expansion, shared by the passes of the complete
// solve (solver.cuh) and by the interaction kernel's fused L2L epilogue (kernels.cuh).
#pragma once

#include <cuda_runtime.h>

namespace octo {

// unique-component index of a symmetric rank-2 / rank-3 tensor, lexicographic order.  Non-recursive on
// purpose: in fully unrolled loops the compiler folds them to constants (a recursive constexpr is called at run
// time in device code and turns every tensor into a local-memory array).
__host__ __device__ __forceinline__ constexpr int u2(int i, int j)
{
    return (i < j ? i : j) * 3 - ((i < j ? i : j) * ((i < j ? i : j) - 1)) / 2 + ((i < j ? j : i) - (i < j ? i : j));
}
__host__ __device__ __forceinline__ constexpr int u3(int i, int j, int k)
{
    // a <= b <= c the sorted indices
    return u2((i + j + k) - (i < j ? (i < k ? i : k) : (j < k ? j : k)) - (i > j ? (i > k ? i : k) : (j > k ? j : k)),
              (i > j ? (i > k ? i : k) : (j > k ? j : k))) +
           ((i < j ? (i < k ? i : k) : (j < k ? j : k)) == 0 ? 0 : ((i < j ? (i < k ? i : k) : (j < k ? j : k)) == 1 ? 3 : 4));
}
static_assert(u2(0, 0) == 0 && u2(1, 0) == 1 && u2(0, 2) == 2 && u2(1, 1) == 3 && u2(2, 1) == 4 && u2(2, 2) == 5, "u2");
static_assert(u3(0, 0, 0) == 0 && u3(0, 1, 0) == 1 && u3(2, 0, 0) == 2 && u3(1, 0, 1) == 3 && u3(2, 1, 0) == 4 &&
              u3(0, 2, 2) == 5 && u3(1, 1, 1) == 6 && u3(1, 2, 1) == 7 && u3(2, 1, 2) == 8 && u3(2, 2, 2) == 9, "u3");

// Taylor shift of a parent expansion L (20 unique components in registers) by e, orders 0..NORD:
//   out3 = L3;  out2_ij = L2_ij + L3_ijk e_k;  out1_i = L1_i + L2_ij e_j + 1/2 L3_ijk e_j e_k;
//   out0 = L0 + L1_i e_i + 1/2 L2_ij e_i e_j + 1/6 L3_ijk e_i e_j e_k
// evaluated through the contractions w_ij = L3_ijk e_k, v_i = L2_ij e_j, u_i = w_ij e_j (about 50 FMAs).
template <int NORD>
__device__ __forceinline__ void taylor_shift(const double (&L)[20], const double (&e)[3], double (&out)[20])
{
    double w[6], v[3], u[3];
#pragma unroll
    for (int x = 0; x < 3; ++x)
#pragma unroll
        for (int y = x; y < 3; ++y) {
            double t = 0.0;
#pragma unroll
            for (int z = 0; z < 3; ++z) t = fma(L[10 + u3(x, y, z)], e[z], t);
            w[u2(x, y)] = t;
        }
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        double tv = 0.0, tu = 0.0;
#pragma unroll
        for (int y = 0; y < 3; ++y) {
            tv = fma(L[4 + u2(x, y)], e[y], tv);
            tu = fma(w[u2(x, y)], e[y], tu);
        }
        v[x] = tv;
        u[x] = tu;
    }
    double s0 = L[0];
#pragma unroll
    for (int x = 0; x < 3; ++x) {
        out[1 + x] = L[1 + x] + v[x] + 0.5 * u[x];
        s0 = fma(e[x], L[1 + x] + 0.5 * v[x] + (1.0 / 6.0) * u[x], s0);
    }
    out[0] = s0;
    if (NORD >= 2) {
#pragma unroll
        for (int t = 0; t < 6; ++t) out[4 + t] = L[4 + t] + w[t];
#pragma unroll
        for (int t = 10; t < 20; ++t) out[t] = L[t];
    }
}

}  // namespace octo
