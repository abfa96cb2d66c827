// pty_kernels128.cuh -- forward and adjoint bodies for N = 128 on the register-resident FFT
// (pty_fft128.cuh): one CTA of 512 threads per (position b, probe mode m); the wave stays in
// registers through the whole slice chain, every pointwise step of the method runs on registers in
// layout L1 (real space: rows y = 4 n1 + q of column x) or L3 (k space: ky(j), k1x + 8 k2x; pty_fft128.cuh).
//
// Workspace layouts: psi (incident waves) natural [y][x]; Psi (far field) and the kept spectra in
// "thread order" [register][tid] (private to these kernels, perfectly coalesced).
// Same scaling conventions as pty_kernels.cuh (Ex carries 1/N, Mx carries 1/N^2).
#pragma once
#include "pty_fft128.cuh"
#include "pty_kernels.cuh"

namespace pty {

PTY_DEV void setup128(const Cta128& c, const KArgs& A, int b, int& ry, int& rx) {
    setup_factors<128, F128::NT>(c.tid, c.Ey, c.Ex, c.My, c.Mx, c.red, A, b, ry, rx);
    f128_fill_twiddles(c);
    pty_cta_sync();
}

PTY_DEV void block_accumulate128(const Cta128& c, int slot, float v) {
    v = warp_sum(v);
    if (warp_leader()) red_add_shared(c.red + slot, v);
}

// ------------------------------------------------------------------------------ background fetches
// Fetch 32 float2 per thread (rows n1 = 0..31 at stride `stride` float2 from p) into tensor memory
// columns [tm, tm + 64), four rows per tick: tick K parks the rows fetched by tick K - 1 and issues the
// loads of rows 4 K .. 4 K + 3.  The rows of the last tick stay in `buf` (use take<7>()).
template <bool STREAM> struct Fetch32 {
    const float2* p;
    size_t stride;
    unsigned tm;
    float2 buf[4];
    template <int K> PTY_DEV void tick() {
        if (K > 0) tmem_st4(tm + 8 * (K - 1), buf);
#pragma unroll
        for (int i = 0; i < 4; ++i)
            buf[i] = STREAM ? ld_stream2_pinned(p + (size_t)(4 * K + i) * stride) : ldg2_pinned(p + (size_t)(4 * K + i) * stride);
    }
    // rows 4 K .. 4 K + 3 (after the transform that ran the ticks; tmem_wait_st() once before the first)
    template <int K> PTY_DEV void take(float2 (&o)[4]) {
        if (K < 7) { tmem_ld4(tm + 8 * K, o); tmem_wait_ld(); }
        else {
#pragma unroll
            for (int i = 0; i < 4; ++i) o[i] = buf[i];
        }
    }
};

// ------------------------------------------------------------------------------ forward (a2-a5)
PTY_DEV void fwd_body128(const KArgs& A, const Cta128& c, int item) {
    constexpr int N = 128;
    const int b = item / A.M, m = item % A.M;
    int ry, rx;
    setup128(c, A, b, ry, rx);
    const size_t NN = (size_t)N * N;
    const size_t bm = (size_t)b * A.M + m;
    const int q = c.q(), x = c.x(), k1x = c.k1x();
    float2 v[32];
    // a3: the object rows of slice s are fetched during the inverse transform that precedes their use
    Fetch32<false> fo;
    fo.p = A.object + ((size_t)ry + q) * A.W + rx + x;
    fo.stride = (size_t)4 * A.W;
    fo.tm = c.tm;
    {   // a2: psi_0 = F^-1[E . P^]   (L3 -> L1)
        const float2* Ph = A.probe_hat + (size_t)m * NN;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int ky = c.ky(j);
            const float2 ey = c.Ey[ky];
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) {
                const int kx = k1x + 8 * k2;
                v[16 * j + k2] = cmul(cmul(ldg2(Ph + ky * N + kx), ey), c.Ex[kx]);
            }
        }
        f128_inverse<0>(c, v, fo);
    }
    for (int s = 0; s < A.Nz; ++s) {
        {   // a3 + a4 (L1): keep psi_{s-1}, phi_s = O_b[s] psi_{s-1}
            float2* save = A.ws_psi + (bm * A.Nz + s) * NN + q * N + x;
            tmem_wait_st();
#define PTY_OBJ_CHUNK(K)                                                   \
            {                                                              \
                float2 o[4];                                               \
                fo.template take<K>(o);                                    \
                _Pragma("unroll") for (int i = 0; i < 4; ++i) {            \
                    st_stream2(save + 4 * (4 * K + i) * N, v[4 * K + i]);  \
                    v[4 * K + i] = cmul(v[4 * K + i], o[i]);               \
                }                                                          \
            }
            PTY_OBJ_CHUNK(7) PTY_OBJ_CHUNK(0) PTY_OBJ_CHUNK(1) PTY_OBJ_CHUNK(2)
            PTY_OBJ_CHUNK(3) PTY_OBJ_CHUNK(4) PTY_OBJ_CHUNK(5) PTY_OBJ_CHUNK(6)
#undef PTY_OBJ_CHUNK
            fo.p += (size_t)A.H * A.W;
        }
        f128_forward(c, v);
        if (s == A.Nz - 1) break;
        {   // a4 (L3): k_x factor of the propagator (k_y factor inside the inverse); keep the spectrum
            float2* hat = A.save_hat ? A.ws_hat + (bm * (A.Nz - 1) + s) * NN + c.tid : nullptr;
#pragma unroll
            for (int r = 0; r < 32; ++r) {
                v[r] = cmul(v[r], c.Mx[k1x + 8 * (r & 15)]);
                if (hat) st_stream2(hat + r * F128::NT, v[r]);
            }
        }
        f128_inverse<+1>(c, v, fo);
    }
    // a5 (L3): Psi = F[phi_Nz] / N, I += |Psi|^2
    float2* Psi = A.ws_Psi + bm * NN + c.tid;
    float* Ib = A.I + (size_t)b * NN;
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const float2 p = cscale(v[r], 1.0f / N);
        st_stream2(Psi + r * F128::NT, p);
        red_add(Ib + c.ky(r >> 4) * N + k1x + 8 * (r & 15), p.x * p.x + p.y * p.y);
    }
}

// ------------------------------------------------------------------------------ adjoint (a7-a13)
PTY_DEV void bwd_body128(const KArgs& A, const Cta128& c, int item) {
    constexpr int N = 128;
    const int b = item / A.M, m = item % A.M;
    int ry, rx;
    setup128(c, A, b, ry, rx);
    const size_t NN = (size_t)N * N;
    const size_t bm = (size_t)b * A.M + m;
    const int q = c.q(), x = c.x(), k1x = c.k1x();
    float2 v[32];
    {   // a7, a8 (L3): g_Psi = 2 (1 - a / sqrt(I)) Psi, g_phi = F^-1[g_Psi]
        const float2* Psi = A.ws_Psi + bm * NN + c.tid;
        const float* Ib = A.I + (size_t)b * NN;
        const float* ab = A.meas + (size_t)b * NN;
#pragma unroll
        for (int h = 0; h < 32; h += 8) {
            float iv[8], av[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int r = h + i, idx = c.ky(r >> 4) * N + k1x + 8 * (r & 15);
                v[r] = ld_stream2(Psi + r * F128::NT);
                iv[i] = ldg1(Ib + idx);
                av[i] = ldg1(ab + idx);
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float w = iv[i] > 1e-30f ? 2.0f * (1.0f - av[i] * rsqrt_f(iv[i])) * (1.0f / N) : 0.f;
                v[h + i] = cscale(v[h + i], w);
            }
        }
        f128_inverse<0>(c, v);
    }
    float acc_ky = 0.f, acc_kx = 0.f, acc_k2 = 0.f;
    for (int s = A.Nz - 1; s >= 0; --s) {
        {   // a9, a10 (L1): g_object patch += conj(psi_{s-1}) g;  g <- conj(O_b[s]) g
            const size_t off = ((size_t)s * A.H + ry + q) * A.W + rx + x;
            const float2* obj = A.object + off;
            float2* gobj = A.g_object + off;
            const float2* psi = A.ws_psi + (bm * A.Nz + s) * NN + q * N + x;
#pragma unroll
            for (int h = 0; h < 32; h += 8) {
                float2 ps[8], o[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    ps[i] = ld_stream2(psi + 4 * (h + i) * N);
                    o[i] = ldg2(obj + (size_t)(4 * (h + i)) * A.W);
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    red_add2(gobj + (size_t)(4 * (h + i)) * A.W, cmulc(ps[i], v[h + i]));
                    v[h + i] = cmulc(o[i], v[h + i]);
                }
            }
        }
        f128_forward(c, v);
        if (s == 0) break;
        {   // a9, a13 (L3): D-sums against the kept spectrum, then conj(Mx) (conj(My) inside the inverse)
            if (A.save_hat) {
                const float2* hat = A.ws_hat + (bm * (A.Nz - 1) + (s - 1)) * NN + c.tid;
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int ky = c.ky(j);
                    const float2 my = c.My[ky];
                    const float kyf = kp_of<N>(ky);
#pragma unroll
                    for (int k2 = 0; k2 < 16; ++k2) {
                        const int r = 16 * j + k2;
                        const float2 hs = cmul(my, ld_stream2(hat + r * F128::NT));
                        const float d = hs.x * v[r].y - hs.y * v[r].x;          // Im(conj(psi^) g^)
                        const float kxf = kp_of<N>(k1x + 8 * k2);
                        acc_ky += d * kyf;
                        acc_kx += d * kxf;
                        acc_k2 += d * (kyf * kyf + kxf * kxf);
                    }
                }
            }
#pragma unroll
            for (int r = 0; r < 32; ++r) v[r] = cmulc(c.Mx[k1x + 8 * (r & 15)], v[r]);
        }
        f128_inverse<-1>(c, v);
    }
    // a11, a12 (L3): g^_0 = F[g_psi0]; probe-gradient accumulation and the position gradient
    const float2* Ph = A.probe_hat + (size_t)m * NN;
    float2* GP = A.GP_hat + (size_t)m * NN;
    float accy = 0.f, accx = 0.f;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const int ky = c.ky(j);
        const float2 ey = c.Ey[ky];
        const float kyf = kp_of<N>(ky);
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) {
            const int kx = k1x + 8 * k2;
            const float2 g = v[16 * j + k2];
            const float2 e = cmul(ey, c.Ex[kx]);                     // E / N
            red_add2(GP + ky * N + kx, cmulc(e, g));
            const float2 ep = cmul(e, ldg2(Ph + ky * N + kx));
            const float t = g.x * ep.y - g.y * ep.x;                 // Im(conj(g^_0) E P^)
            accy += kyf * t;
            accx += kp_of<N>(kx) * t;
        }
    }
    block_accumulate128(c, 0, accy);
    block_accumulate128(c, 1, accx);
    if (A.save_hat) {
        block_accumulate128(c, 2, acc_ky);
        block_accumulate128(c, 3, acc_kx);
        block_accumulate128(c, 4, acc_k2);
    }
    pty_cta_sync();
    if (c.tid == 0) {
        const float two_pi = 6.283185307179586f;
        if (A.g_pos) {
            red_add(A.g_pos + 2 * b, two_pi * c.red[0]);
            red_add(A.g_pos + 2 * b + 1, two_pi * c.red[1]);
        }
        if (A.save_hat) {
            red_add(A.dsum + 4 * b, c.red[2]);
            red_add(A.dsum + 4 * b + 1, c.red[3]);
            red_add(A.dsum + 4 * b + 2, c.red[4]);
        }
    }
}

}  // namespace pty
