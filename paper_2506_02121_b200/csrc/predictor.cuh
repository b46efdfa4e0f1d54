// predictor.cuh — seed of a continued row from the chain's last rows (R18; "the roots at
// phi_j are initial guesses for phi_{j+1}").  Product path only.
//
// One step ahead, the polynomial through the last p + 1 rows equals the sum of the BACKWARD DIFFERENCES at the newest row,
//   z_pred = v_1 + D^1 v_1 + D^2 v_1 + ... + D^p v_1,     D^1 v_1 = v_1 - v_2,  D^(j+1) = D(D^j),
// so the order can be chosen root by root: term j is added only while the terms still fall by at least a factor two
// from one order to the next.  On a smooth chain they fall by ~ dphi / (scale of the motion) per order until they reach
// the rounding of the stored rows (where they start to double: those terms are noise and are left out).  On a chain
// whose column has swapped between two nearby roots from one row to the next -- it happens where two branches of the
// critical curve pass close to each other -- the first differences do not fall at all and the seed is the previous
// row's root itself (order 0), which pulls the column back onto one root; a fixed high order extrapolated the zig-zag
// instead (seed errors of several theta_star, six iterations per row on every other row of a cfg4 sub-chain).
// Only the starting guess depends on this; the fixed point and the freeze test do not.
#pragma once
#include <cuda_runtime.h>

namespace mlcc {

constexpr int PRED_MAX_ORDER = 8;

// v[0] = newest row (one step behind the row to seed), v[1] the one before, ...; order <= PRED_MAX_ORDER
__device__ __forceinline__ double2 predict_adaptive(const double2 *v, int order)
{
    double2 d[PRED_MAX_ORDER + 1];
    double2 term[PRED_MAX_ORDER + 1];
    double n2[PRED_MAX_ORDER + 2];
#pragma unroll
    for (int q = 0; q <= PRED_MAX_ORDER; ++q) d[q] = q <= order ? v[q] : make_double2(0.0, 0.0);
#pragma unroll
    for (int j = 1; j <= PRED_MAX_ORDER; ++j) {
#pragma unroll
        for (int q = 0; q + j <= PRED_MAX_ORDER; ++q) {
            d[q].x -= d[q + 1].x;
            d[q].y -= d[q + 1].y;
        }
        term[j] = d[0];
        n2[j] = d[0].x * d[0].x + d[0].y * d[0].y;
    }
    double2 z = v[0];
#pragma unroll
    for (int j = 1; j <= PRED_MAX_ORDER; ++j) {
        if (j > order) break;
        if (!(j == order || n2[j + 1] <= 0.25 * n2[j])) break;
        z.x += term[j].x;
        z.y += term[j].y;
    }
    return z;
}

}  // namespace mlcc
