// pty_kernels128.cuh -- N = 128 helpers on the one-item register-resident FFT (pty_fft128.cuh):
// a0: the probe spectrum P^ = F[P] / N written in the thread order of the two-items-per-CTA kernels
// (layout K: [register r][tid = 128 o + ky], register r of role o holds k_x = 8 o + (r & 7) + 32 (r >> 3));
// a11: g_probe = F^-1[G^_P] / N read from the same order.  One CTA of 512 threads per probe mode, once per call.
#pragma once
#include "pty_fft128.cuh"
#include "pty_kernels.cuh"

namespace pty {

// ------------------------------------------------------------------------------ a0 / a11 helpers
// P^_t[m] = F[P[m]] / N in thread order (one CTA per mode)
PTY_DEV void probe_hat_body128(const float2* probe, float2* probe_hat_t, const Cta128& c, int m) {
    constexpr int N = 128;
    f128_fill_twiddles(c);
    pty_cta_sync();
    const float2* src = probe + (size_t)m * N * N + c.g() * N + c.cc();
    float2 v[32];
#pragma unroll
    for (int n = 0; n < 32; ++n) v[n] = ldg2(src + 4 * n * N);
    f128_forward(c, v);
    float2* dst = probe_hat_t + (size_t)m * N * N + c.tid;
#pragma unroll
    for (int r = 0; r < 32; ++r) dst[r * F128::NT] = cscale(v[r], 1.0f / N);
}

// g_probe[m] (+)= F^-1[G^_P_t[m]] / N (one CTA per mode)
PTY_DEV void probe_grad_body128(const float2* GP_t, float2* g_probe, int accumulate, const Cta128& c, int m) {
    constexpr int N = 128;
    f128_fill_twiddles(c);
    pty_cta_sync();
    const float2* src = GP_t + (size_t)m * N * N + c.tid;
    float2 v[32];
#pragma unroll
    for (int r = 0; r < 32; ++r) v[r] = src[r * F128::NT];
    f128_inverse(c, v);
    float2* dst = g_probe + (size_t)m * N * N + c.g() * N + c.cc();
#pragma unroll
    for (int n = 0; n < 32; ++n) {
        float2 o = cscale(v[n], 1.0f / N);
        if (accumulate) o = cadd(o, dst[4 * n * N]);
        dst[4 * n * N] = o;
    }
}

}  // namespace pty
