// ann_common.cuh -- the per-cell prologue (x = {T, p, F(Y)}, Z-score) and epilogue
// (A9-A11, A17: inverse Box-Cox in its expm1/log1p form, sum-to-one renormalisation, density,
// source term) shared by the fp32 (ann_fp32.cu) and bf16/tcgen05 (ann_bf16.cu) MLP kernels.
#pragma once
#include "common.cuh"

// Box-Cox feature of one mass fraction, z-scored:  ((y^lambda - 1)/lambda - mean) / std.
__device__ __forceinline__ float ann_feature_Y(float y, float lambda, float inv_lambda, float mean, float inv_std) {
    const float q = powf(y, lambda);  // powf(0, lambda) = 0 -> F(0) = -1/lambda (A10)
    return ((q - 1.0f) * inv_lambda - mean) * inv_std;
}

// Change of Y_k before renormalisation, dY*_k = Y*_k - Y_k with
//   Y*_k = max(Y_k^lambda + lambda Delta_k, 0)^(1/lambda)
// written as Y_k expm1(log1p(lambda Delta_k Y_k^-lambda)/lambda): no cancellation for small Delta.
__device__ __forceinline__ float ann_dystar(float y, float delta, float lambda, float inv_lambda) {
    if (y > 0.f) {
        const float q = powf(y, lambda);
        const float z = lambda * delta / q;
        if (!(z > -1.0f)) return -y;  // base <= 0 -> Y* = 0
        return y * expm1f(log1pf(z) * inv_lambda);
    }
    const float base = lambda * delta;
    return base > 0.f ? powf(base, inv_lambda) : 0.f;
}

// Second half of the epilogue for one species once the two sums are known:
//   S - 1 = (sum_j Y_j - 1) + sum_j dY*_j;   dY_k = Y*_k/S - Y_k = (dY*_k - Y_k (S - 1))/S.
__device__ __forceinline__ float ann_renorm_dY(float dystar, float y, double Sm1, double inv_S) {
    return (float)(((double)dystar - (double)y * Sm1) * inv_S);
}

// exact GELU x Phi(x) (A13), Phi through erfc so that x << 0 does not cancel
__device__ __forceinline__ float gelu_erf(float x) { return 0.5f * x * erfcf(-0.70710678118654752f * x); }
