// pppm_common.cuh -- pieces shared by pppm.cu and pppm_sweep.cu (PAPER.md II.F; reading S10).
#pragma once

// centred cardinal B-spline of order 5 on mesh offsets -2..2 (reading S10); dx = u - round(u) in [-1/2, 1/2)
__device__ __forceinline__ void bspline5(float dx, float* __restrict__ w)
{
    const float d2 = dx * dx, d3 = d2 * dx, d4 = d2 * d2;
    w[0] = (1.f - 8.f * dx + 24.f * d2 - 32.f * d3 + 16.f * d4) * (1.f / 384.f);
    w[1] = (19.f - 44.f * dx + 24.f * d2 + 16.f * d3 - 16.f * d4) * (1.f / 96.f);
    w[2] = (115.f - 120.f * d2 + 48.f * d4) * (1.f / 192.f);
    w[3] = (19.f + 44.f * dx + 24.f * d2 - 16.f * d3 - 16.f * d4) * (1.f / 96.f);
    w[4] = (1.f + 8.f * dx + 24.f * d2 + 32.f * d3 + 16.f * d4) * (1.f / 384.f);
}
