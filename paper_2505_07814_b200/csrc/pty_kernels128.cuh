// pty_kernels128.cuh -- forward and adjoint bodies for N = 128 on the register-resident FFT
// (pty_fft128.cuh): one CTA of 512 threads per (position b, probe mode m); the wave stays in
// registers through the whole slice chain, every pointwise step of the method runs on registers in
// layout R (real space: rows y = 4 n1 + q of column x = c) or layout K (k space: row ky = c,
// columns kx = 8 g + i + 32 k2 in register 8 k2 + i).
//
// Workspace layouts: psi (incident waves) in layout-R thread order as 16-byte pairs, [n1 / 2][tid] float4 =
// (v[n1], v[n1 + 1]) -- written and read with one 16-byte access per two rows; every k-space array private to these
// kernels (P^, Psi, the kept spectra, the seed weights, G^_P) in "thread order" [register][tid], which
// is perfectly coalesced in layout K.  Same scaling conventions as pty_kernels.cuh (Ex carries 1/N,
// Mx carries 1/N^2).
#pragma once
#ifndef PTY_BWD_SPLIT
#define PTY_BWD_SPLIT 0
#endif
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
// Fetch 32 float2 per thread (rows n1 = 0..31 at stride `stride` float2 from p) into the tensor-memory
// staging block, four rows per tick: tick K (0..7) issues the loads of rows 4 K .. 4 K + 3, tick K + 1
// parks them.  Nine ticks: everything is parked before the inverse transform's last exchange.
// STREAM: the source is a saved wave in thread order (p = the thread's first float4, stride in float4 between pairs).
// Two schedules: tick<K> puts all eight chunks into one inverse transform (the first slice of an item);
// tick_fwd<K> / tick_inv<K> spread them over the forward transform that precedes the inverse (chunks 0-3, one
// every three ticks) and the inverse itself (chunks 4-7, one every two ticks), which doubles the time between
// a load and its park.  The staging block is free during the forward transform: its previous content was consumed
// by the pointwise step just before.
template <bool STREAM> struct Fetch32 {
    const float2* p;
    size_t stride;
    unsigned tm;
    bool on;
    float2 buf[4];
    template <int C> PTY_DEV void issue() {
        if (STREAM) {
            const float4* p4 = reinterpret_cast<const float4*>(p);
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const float4 t = ld_stream4_pinned(p4 + (size_t)(2 * C + i) * stride);
                buf[2 * i] = make_float2(t.x, t.y);
                buf[2 * i + 1] = make_float2(t.z, t.w);
            }
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) buf[i] = ldg2_pinned(p + (size_t)(4 * C + i) * stride);
        }
    }
    template <int C> PTY_DEV void park() { tmem_st4(tm + 8 * C, buf); }
    template <int K> PTY_DEV void tick() {
        if (K > 0 && K <= 8) park<(K > 0 && K <= 8) ? K - 1 : 0>();
        if (K < 8) issue<K < 8 ? K : 0>();
    }
    template <int K> PTY_DEV void tick_fwd() {
        if (!on) return;
        if (K == 3 || K == 6 || K == 9 || K == 12) park<(K % 3 == 0 && K >= 3) ? K / 3 - 1 : 0>();
        if (K == 0 || K == 3 || K == 6 || K == 9) issue<(K % 3 == 0 && K <= 9) ? K / 3 : 0>();
    }
    template <int K> PTY_DEV void tick_inv() {
        if (K == 2 || K == 4 || K == 6 || K == 8) park<(K % 2 == 0 && K >= 2) ? 3 + K / 2 : 0>();
        if (K == 0 || K == 2 || K == 4 || K == 6) issue<(K % 2 == 0 && K <= 6) ? 4 + K / 2 : 0>();
    }
    // rows 4 K .. 4 K + 3 (tmem_wait_st() once before the first take)
    template <int K> PTY_DEV void take(float2 (&o)[4]) { tmem_ld4(tm + 8 * K, o); tmem_wait_ld(); }
};

template <class F> struct FetchFwdHalf { F& f; template <int K> PTY_DEV void tick() { f.template tick_fwd<K>(); } };
template <class F> struct FetchInvHalf { F& f; template <int K> PTY_DEV void tick() { f.template tick_inv<K>(); } };

// Fetch 32 float2 per thread into the EXCHANGE block while it is free (after a FREE exchange), eight rows
// per tick of the last fft32 of the inverse transform: ticks 0..3 issue rows 8 J .. 8 J + 7, ticks 1, 2, 3
// and 5 park them.
struct Fetch32x8 {
    const float2* p;
    size_t stride;
    unsigned tm;
    float2 buf[8];
    template <int J> PTY_DEV void tick() {
        if (J >= 1 && J <= 3) tmem_st8r(tm + 16 * (J - 1), buf);
        if (J == 5) tmem_st8r(tm + 48, buf);
        if (J <= 3) {
#pragma unroll
            for (int i = 0; i < 8; ++i) buf[i] = ldg2_pinned(p + (size_t)(8 * J + i) * stride);
        }
    }
    template <int J> PTY_DEV void take(float2 (&o)[8]) { tmem_ld8r(tm + 16 * J, o); tmem_wait_ld(); }
};

// ------------------------------------------------------------------------------ forward (a2-a5)
PTY_DEV void fwd_body128(const KArgs& A, const Cta128& c, int item) {
    constexpr int N = 128;
    const int b = item / A.M, m = item % A.M;
    int ry, rx;
    setup128(c, A, b, ry, rx);
    const size_t NN = (size_t)N * N;
    const size_t bm = (size_t)b * A.M + m;
    const int g = c.g(), cc = c.cc();
    float2 v[32];
    // a3: the object rows of slice s are fetched during the inverse transform that precedes their use
    Fetch32<false> fo;
    fo.p = A.object + ((size_t)ry + g) * A.W + rx + cc;
    fo.stride = (size_t)4 * A.W;
    fo.tm = c.tm_s();
    fo.on = true;
    FetchFwdHalf<Fetch32<false>> fo_fwd{fo};
    FetchInvHalf<Fetch32<false>> fo_inv{fo};
    NoBg nobg;
    {   // a2: psi_0 = F^-1[E . P^]   (K -> R)
        const float2* Ph = A.probe_hat + (size_t)m * NN + c.tid;
        const float2 ey = c.Ey[cc];
#pragma unroll
        for (int r = 0; r < 32; ++r) v[r] = cmul(cmul(ldg2(Ph + r * F128::NT), ey), c.Ex[c.kx(r)]);
        f128_inverse<false>(c, v, fo, nobg);
    }
    for (int s = 0; s < A.Nz; ++s) {
        {   // a3 + a4 (R): keep psi_{s-1}, phi_s = O_b[s] psi_{s-1}
            float4* save = reinterpret_cast<float4*>(A.ws_psi + (bm * A.Nz + s) * NN) + c.tid;
            tmem_wait_st();
#define PTY_OBJ_CHUNK(K)                                                   \
            {                                                              \
                float2 o[4];                                               \
                fo.template take<K>(o);                                    \
                st_stream4(save + (2 * K) * F128::NT, v[4 * K], v[4 * K + 1]);          \
                st_stream4(save + (2 * K + 1) * F128::NT, v[4 * K + 2], v[4 * K + 3]);  \
                _Pragma("unroll") for (int i = 0; i < 4; ++i)              \
                    v[4 * K + i] = cmul(v[4 * K + i], o[i]);               \
            }
            PTY_OBJ_CHUNK(0) PTY_OBJ_CHUNK(1) PTY_OBJ_CHUNK(2) PTY_OBJ_CHUNK(3)
            PTY_OBJ_CHUNK(4) PTY_OBJ_CHUNK(5) PTY_OBJ_CHUNK(6) PTY_OBJ_CHUNK(7)
#undef PTY_OBJ_CHUNK
            fo.p += (size_t)A.H * A.W;
        }
        fo.on = s < A.Nz - 1;
        f128_forward<true>(c, v, fo_fwd);
        if (s == A.Nz - 1) break;
        {   // a4 (K): propagator M = My[ky] Mx[kx] (/N^2); keep the spectrum F[psi_s]
            float2* hat = A.save_hat ? A.ws_hat + (bm * (A.Nz - 1) + s) * NN + c.tid : nullptr;
            const float2 my = c.My[cc];
#pragma unroll
            for (int r = 0; r < 32; ++r) {
                v[r] = cmul(v[r], cmul(my, c.Mx[c.kx(r)]));
                if (hat) st_stream2(hat + r * F128::NT, v[r]);
            }
        }
        f128_inverse<false>(c, v, fo_inv, nobg);
    }
    // a5 (K): Psi = F[phi_Nz] / N, I += |Psi|^2 (transposed through X so that the reductions into the
    // natural [ky][kx] array are coalesced)
    float2* Psi = A.ws_Psi + bm * NN + c.tid;
    float* Xf = reinterpret_cast<float*>(c.X);
    pty_cta_sync();                                   // every thread is done with the last transpose
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const float2 p = cscale(v[r], 1.0f / N);
        st_stream2(Psi + r * F128::NT, p);
        Xf[cc * F128::P + c.kx(r)] = p.x * p.x + p.y * p.y;
    }
    pty_cta_sync();
    float* Ib = A.I + (size_t)b * NN;
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const int idx = j * F128::NT + c.tid;
        red_add(Ib + idx, Xf[(idx >> 7) * F128::P + (idx & 127)]);
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
    const int g = c.g(), cc = c.cc();
    float2 v[32];
    // a9: the saved waves psi_{s-1} and the object rows O_b[s] of slice s are fetched during the inverse
    // transform that precedes their use: psi (HBM stream) over its 9 ticks into the staging block, the
    // object rows over the last fft32 into the exchange block once it is free.
    Fetch32<true> fp;
    fp.p = A.ws_psi + (bm * A.Nz + (A.Nz - 1)) * NN + 2 * c.tid;
    fp.stride = F128::NT;
    fp.tm = c.tm_s();
    fp.on = true;
    FetchFwdHalf<Fetch32<true>> fp_fwd{fp};
    FetchInvHalf<Fetch32<true>> fp_inv{fp};
    Fetch32x8 fo;
    fo.p = A.object + ((size_t)(A.Nz - 1) * A.H + ry + g) * A.W + rx + cc;
    fo.stride = (size_t)4 * A.W;
    fo.tm = c.tm_x();
    NoBg nobg;
    {   // a7, a8 (K): g_Psi = w Psi with the seed weights w = 2 (1 - a / sqrt(I)) / N, g_phi = F^-1[g_Psi]
        const float2* Psi = A.ws_Psi + bm * NN + c.tid;
        const float* Wt = A.seed_w + (size_t)b * NN + c.tid;
#pragma unroll
        for (int h = 0; h < 32; h += 8) {
            float wv[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                v[h + i] = ld_stream2(Psi + (h + i) * F128::NT);
                wv[i] = ldg1(Wt + (h + i) * F128::NT);
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) v[h + i] = cscale(v[h + i], wv[i]);
        }
        f128_inverse<true>(c, v, fp, fo);
    }
    float acc_ky = 0.f, acc_kx = 0.f, acc_k2 = 0.f;
    for (int s = A.Nz - 1; s >= 0; --s) {
        {   // a9, a10 (R): g_object patch += conj(psi_{s-1}) g;  g <- conj(O_b[s]) g
            float2* gobj = A.g_object + ((size_t)s * A.H + ry + g) * A.W + rx + cc;
            tmem_wait_st();
#define PTY_BWD_CHUNK(J)                                                                              \
            {                                                                                         \
                float2 o[8], pa[4], pb[4];                                                            \
                fo.template take<J>(o);                                                               \
                fp.template take<2 * J>(pa);                                                          \
                fp.template take<2 * J + 1>(pb);                                                      \
                _Pragma("unroll") for (int i = 0; i < 8; ++i) {                                       \
                    const float2 ps = i < 4 ? pa[i & 3] : pb[i & 3];                                  \
                    red_add2(gobj + (size_t)(4 * (8 * J + i)) * A.W, cmulc(ps, v[8 * J + i]));       \
                    v[8 * J + i] = cmulc(o[i], v[8 * J + i]);                                         \
                }                                                                                     \
            }
            PTY_BWD_CHUNK(0) PTY_BWD_CHUNK(1) PTY_BWD_CHUNK(2) PTY_BWD_CHUNK(3)
#undef PTY_BWD_CHUNK
            fp.p -= (size_t)N * N;
            fo.p -= (size_t)A.H * A.W;
        }
#if PTY_BWD_SPLIT
        fp.on = s > 0;
        f128_forward<false>(c, v, fp_fwd);
#else
        f128_forward<false>(c, v, nobg);
#endif
        if (s == 0) break;
        {   // a9, a13 (K): D-sums against the kept spectrum, then conj(M)
            const float2 my = c.My[cc];
            if (A.save_hat) {
                const float2* hat = A.ws_hat + (bm * (A.Nz - 1) + (s - 1)) * NN + c.tid;
                const float kyf = kp_of<N>(cc);
#pragma unroll
                for (int r = 0; r < 32; ++r) {
                    const float2 hs = ld_stream2(hat + r * F128::NT);
                    const float d = hs.x * v[r].y - hs.y * v[r].x;          // Im(conj(psi^) g^)
                    const float kxf = kp_of<N>(c.kx(r));
                    acc_ky += d * kyf;
                    acc_kx += d * kxf;
                    acc_k2 += d * (kyf * kyf + kxf * kxf);
                }
            }
#pragma unroll
            for (int r = 0; r < 32; ++r) v[r] = cmulc(cmul(my, c.Mx[c.kx(r)]), v[r]);
        }
#if PTY_BWD_SPLIT
        f128_inverse<true>(c, v, fp_inv, fo);
#else
        f128_inverse<true>(c, v, fp, fo);
#endif
    }
    // a11, a12 (K): g^_0 = F[g_psi0]; probe-gradient accumulation and the position gradient
    const float2* Ph = A.probe_hat + (size_t)m * NN + c.tid;
    float2* GP = A.GP_hat + (size_t)m * NN + c.tid;
    float accy = 0.f, accx = 0.f;
    {
        const float2 ey = c.Ey[cc];
        const float kyf = kp_of<N>(cc);
#pragma unroll
        for (int r = 0; r < 32; ++r) {
            const int kx = c.kx(r);
            const float2 gg = v[r];
            const float2 e = cmul(ey, c.Ex[kx]);                     // E / N
            red_add2(GP + r * F128::NT, cmulc(e, gg));
            const float2 ep = cmul(e, ldg2(Ph + r * F128::NT));
            const float t = gg.x * ep.y - gg.y * ep.x;               // Im(conj(g^_0) E P^)
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
