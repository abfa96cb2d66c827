// pty_fft128.cuh -- register-resident 128 x 128 2-D FFT for one CTA of 512 threads on sm_100a:
// ONE shared-memory exchange per 2-D FFT; the other two exchanges go through tensor memory (TMEM).
//
// The wave lives in registers, 32 complex values per thread.  Thread id = 128 g + c (g < 4, c < 128).
// A 1-D FFT of length 128 along one axis is split 128 = 32 x 4 (decimation in time):
//   (a) radix-32 in registers over the 32 strided samples a thread holds,
//   (b) an exchange among the FOUR threads that share c (they differ in g only),
//   (c) twiddle W128^(q k1) and radix-4 over q in registers.
// The four threads of (b) are the same lane of the four warps of one SM sub-partition, i.e. they
// share one TMEM lane: each writes its 32 values to its own 64 TMEM columns (tcgen05.st) and reads
// 8 values from each of the four column blocks (tcgen05.ld).  That exchange costs no shared-memory
// bandwidth and does not go through the LSU pipe; its barrier covers the 4 warps of one sub-partition.
// Between the two axes the wave is transposed through shared memory, in place: element (ky, x) has
// the single home slot X[ky * 129 + x]; the y-side thread (g, x) touches it with lanes along x, the
// x-side thread (g, ky) with lanes along ky (stride 129 float2: conflict-free), and a slot is never
// touched by two threads between two CTA barriers.  A forward transform and its inverse are exact
// mirrors, so a chain  F^-1 -> (pointwise, layout R) -> F -> (pointwise, layout K) -> F^-1 ...  needs one
// CTA barrier and two or three sub-partition barriers per 2-D FFT.
//
//   layout R (real space): thread (q = g, x = c)   holds a[y = 4 n1 + q][x]           in v[n1],  n1 < 32
//   layout K (k space):    thread (g, ky = c)      holds A[ky][kx = 8 g + i + 32 k2]  in v[8 k2 + i]
//
//   forward:  fft32 over n1 | T | tw, radix-4 over q -> ky = 8 g + i + 32 k2y | S (transpose) |
//             x = 4 n1x + xq: fft32 over n1x | T | tw, radix-4 over xq -> kx = 8 g + i + 32 k2x.
//   inverse:  the same steps conjugated, in reverse order.  Both are unscaled.
//
// TMEM use: 512 columns x 128 lanes, allocated once per CTA.  Thread (g, c) owns lane c, columns
// [128 g, 128 g + 128): the first 64 are the exchange block, the last 64 a staging buffer where the
// kernel bodies park global data fetched early (Fetch32 in pty_kernels128.cuh).
#pragma once
#include "pty_fft.cuh"

namespace pty {

struct F128 {
    static constexpr int N = 128, NT = 512;
    static constexpr int P = 129;              // pitch of X (float2)
    static constexpr size_t xch_bytes = size_t(128) * P * sizeof(float2);
    // tables: twg[4][8][4], Ey, Ex, My, Mx [128 each] (float2), red[64] (float), TMEM base (16 B)
    static constexpr size_t table_bytes = (128 + 4 * 128) * sizeof(float2) + 64 * sizeof(float) + 16;
    static constexpr size_t smem_bytes = xch_bytes + table_bytes;
};

struct Cta128 {
    int tid;
    float2* X;                       // transpose space
    float2* twg;                     // W128^(q (8 g + i)) [g][i][q]   (forward sign)
    float2 *Ey, *Ex, *My, *Mx;       // [128] shift and propagator factors (Ex carries 1/N, Mx 1/N^2)
    float* red;
    unsigned tmq;                    // TMEM address of this thread's lane quarter, column 0
    PTY_DEV int g() const { return tid >> 7; }
    PTY_DEV int cc() const { return tid & 127; }
    PTY_DEV unsigned tm_x() const { return tmq + 128u * (unsigned)(tid >> 7); }          // exchange block
    PTY_DEV unsigned tm_s() const { return tmq + 128u * (unsigned)(tid >> 7) + 64u; }    // staging block
    // layout K: k_x of register r = 8 k2 + i
    PTY_DEV int kx(int r) const { return 8 * (tid >> 7) + (r & 7) + 32 * (r >> 3); }
};

// ---- FMA-form twiddles (cos / sin of 2 pi j / 32 as compile-time constants).  w u = gamma (alpha u + beta (i u)) with |alpha|, |beta| <= 1 and one of them 1: the inner
// bracket u' is ONE packed FMA, and the real scale gamma is carried as "pending" into the add/sub pair that consumes
// the value (y +- gamma u' = two packed FMAs instead of two packed adds): 3 packed instructions per twiddled
// butterfly input instead of 4, and no extra rounding step.  All constants are compile-time.
PTY_DEV constexpr double cd32(int j) {
    constexpr double t[9] = {1.0, 0.98078528040323044913, 0.92387953251128675613, 0.83146961230254523708,
                             0.70710678118654752440, 0.55557023301960222474, 0.38268343236508977173,
                             0.19509032201612826785, 0.0};
    j &= 31;
    return j <= 8 ? t[j] : j <= 16 ? -t[16 - j] : j <= 24 ? -t[j - 16] : t[32 - j];
}
PTY_DEV constexpr double dabs_(double x) { return x < 0 ? -x : x; }
// w = exp(i DIR 2 pi J / 32)
template <int J, int DIR> struct TwC {
    static constexpr int Jm = ((J % 32) + 32) % 32;
    static constexpr double C = cd32(Jm), S = DIR * cd32(Jm - 8);
    static constexpr bool trivial = (Jm % 8 == 0);
    static constexpr bool caseA = dabs_(C) >= dabs_(S);
    static constexpr float gamma = trivial ? 1.0f : (caseA ? (float)C : (float)S);
    static constexpr float T = trivial ? 0.0f : (caseA ? (float)(S / C) : (float)(C / S));
    // u' with w u = gamma u'
    static PTY_DEV float2 prep(float2 u) {
        if constexpr (Jm == 0) return u;
        else if constexpr (Jm == 8) return mul_qi<DIR>(u);
        else if constexpr (Jm == 16) return make_float2(-u.x, -u.y);
        else if constexpr (Jm == 24) return mul_qi<-DIR>(u);
        else if constexpr (caseA) return __ffma2_rn(make_float2(u.y, u.x), make_float2(-T, T), u);
        else return __ffma2_rn(u, make_float2(T, T), make_float2(-u.y, u.x));
    }
};
// y + g x, g a compile-time constant at every call site
PTY_DEV float2 axpy_c(float g, float2 x, float2 y) {
    if (g == 1.0f) return cadd(y, x);
    if (g == -1.0f) return csub(y, x);
    return __ffma2_rn(make_float2(g, g), x, y);
}

// 8-point DFT over n2 of the values W32^(K1 n2) u[n2] (the twiddles are NOT yet applied to u), natural order out.
template <int K1, int DIR> PTY_DEV void fft8_pend(float2 (&w)[8]) {
    using T1 = TwC<K1 * 1, DIR>; using T2 = TwC<K1 * 2, DIR>; using T3 = TwC<K1 * 3, DIR>; using T4 = TwC<K1 * 4, DIR>;
    using T5 = TwC<K1 * 5, DIR>; using T6 = TwC<K1 * 6, DIR>; using T7 = TwC<K1 * 7, DIR>;
    constexpr float g1 = T1::gamma, g2 = T2::gamma, g3 = T3::gamma, g4 = T4::gamma, g5 = T5::gamma, g6 = T6::gamma,
                    g7 = T7::gamma;
    constexpr float h = 0.70710678118654752440f;
    const float2 p1 = T1::prep(w[1]), p2 = T2::prep(w[2]), p3 = T3::prep(w[3]), p4 = T4::prep(w[4]),
                 p5 = T5::prep(w[5]), p6 = T6::prep(w[6]), p7 = T7::prep(w[7]);
    // even half: E_k, clean
    const float2 t0 = axpy_c(g4, p4, w[0]), t1 = axpy_c(-g4, p4, w[0]);
    const float2 pe = axpy_c(g6 / g2, p6, p2), me = mul_qi<DIR>(axpy_c(-(g6 / g2), p6, p2));
    const float2 e0 = axpy_c(g2, pe, t0), e2 = axpy_c(-g2, pe, t0), e1 = axpy_c(g2, me, t1), e3 = axpy_c(-g2, me, t1);
    // odd half: O_k = g1 q_k
    const float2 a = axpy_c(g5 / g1, p5, p1), b = axpy_c(-(g5 / g1), p5, p1);
    const float2 c = axpy_c(g7 / g3, p7, p3), d = mul_qi<DIR>(axpy_c(-(g7 / g3), p7, p3));
    const float2 q0 = axpy_c(g3 / g1, c, a), q2 = mul_qi<DIR>(axpy_c(-(g3 / g1), c, a));
    const float2 q1 = axpy_c(g3 / g1, d, b), q3 = mul_qi<DIR>(axpy_c(-(g3 / g1), d, b));
    const float2 s1 = cadd(q1, mul_qi<DIR>(q1)), s3 = cadd(q3, mul_qi<DIR>(q3));
    w[0] = axpy_c(g1, q0, e0); w[4] = axpy_c(-g1, q0, e0);
    w[2] = axpy_c(g1, q2, e2); w[6] = axpy_c(-g1, q2, e2);
    w[1] = axpy_c(g1 * h, s1, e1); w[5] = axpy_c(-(g1 * h), s1, e1);
    w[3] = axpy_c(g1 * h, s3, e3); w[7] = axpy_c(-(g1 * h), s3, e3);
}

// ---- FMA form of the cross-thread radix-4 stage with its variable twiddles W128^(q gi), q = 1..3 (forward sign):
// W128^(q gi) = g_q (1 + i T_q), so w u = g (u + T (i u)).  A zero cosine (q gi = 32) becomes g = 2^-40, T = -2^40, which
// gives -i u exactly.  Table entry of gi, 12 floats: (-T1, T1, -T2, T2), (-T3, T3, r31, r31), (g2, g2, g1, g1), r31 = g3/g1.
PTY_DEV void fill_twf(int gi, float* e) {
    double g[4], T[4];
    for (int q = 1; q < 4; ++q) {
        double sn, cs;
        sincospi(2.0 * (double)(q * gi) / 128.0, &sn, &cs);
        if ((q * gi) % 64 == 32) cs = 9.094947017729282e-13;
        g[q] = cs; T[q] = -sn / cs;
    }
    e[0] = (float)-T[1]; e[1] = (float)T[1]; e[2] = (float)-T[2]; e[3] = (float)T[2];
    e[4] = (float)-T[3]; e[5] = (float)T[3]; e[6] = e[7] = (float)(g[3] / g[1]);
    e[8] = e[9] = (float)g[2]; e[10] = e[11] = (float)g[1];
}
// (a0, a1, a2, a3) <- forward radix-4 butterfly of (a0, w1 a1, w2 a2, w3 a3): 11 packed FMAs
PTY_DEV void bfly4_tw_fma(float4 A, float4 Bq, float4 Cq, float2& a0, float2& a1, float2& a2, float2& a3) {
    const float2 P1 = make_float2(A.x, A.y), P2 = make_float2(A.z, A.w), P3 = make_float2(Bq.x, Bq.y);
    const float2 R = make_float2(Bq.z, Bq.w), G2s = make_float2(Cq.x, Cq.y), G1s = make_float2(Cq.z, Cq.w);
    const float2 p1 = __ffma2_rn(make_float2(a1.y, a1.x), P1, a1);
    const float2 p2 = __ffma2_rn(make_float2(a2.y, a2.x), P2, a2);
    const float2 p3 = __ffma2_rn(make_float2(a3.y, a3.x), P3, a3);
    const float2 t0 = __ffma2_rn(G2s, p2, a0), t1 = __ffma2_rn(make_float2(-G2s.x, -G2s.y), p2, a0);
    const float2 pp = __ffma2_rn(R, p3, p1);
    const float2 mm = mul_qi<-1>(__ffma2_rn(make_float2(-R.x, -R.y), p3, p1));
    a0 = __ffma2_rn(G1s, pp, t0);
    a2 = __ffma2_rn(make_float2(-G1s.x, -G1s.y), pp, t0);
    a1 = __ffma2_rn(G1s, mm, t1);
    a3 = __ffma2_rn(make_float2(-G1s.x, -G1s.y), mm, t1);
}

// Background work interleaved with a transform: the transforms call bg.tick<K>() at points spread over
// their arithmetic (K = 0, 1, ... in program order); the kernel bodies use the ticks to fetch the global
// data of the NEXT pointwise step in small chunks and park it in tensor memory.  The inverse transform
// has 9 ticks (0..8) before its last TMEM exchange and 6 ticks of a second functor (0..5) after it, when
// the exchange block is free and can serve as a second staging buffer.
struct NoBg { template <int K> PTY_DEV void tick() {} };

// 32-point DFT in registers, natural order in and out.  n = 8 n1 + n2, k = k1 + 4 k2.
// Four ticks TB .. TB + 3: after the first stage and after each of the first three radix-8 groups.
template <int DIR, int TB, class BG> PTY_DEV void fft32(float2 (&v)[32], BG& bg) {
#pragma unroll
    for (int n2 = 0; n2 < 8; ++n2) bfly4<DIR>(v[n2], v[8 + n2], v[16 + n2], v[24 + n2]);   // -> v[8 k1 + n2]
    bg.template tick<TB>();
    {
        float2 o[32];
#define PTY_F8(K1)                                                                         \
        {                                                                                  \
            float2 w[8];                                                                   \
            _Pragma("unroll") for (int n2 = 0; n2 < 8; ++n2) w[n2] = v[8 * K1 + n2];       \
            fft8_pend<K1, DIR>(w);                                                         \
            _Pragma("unroll") for (int k2 = 0; k2 < 8; ++k2) o[K1 + 4 * k2] = w[k2];       \
        }
        PTY_F8(0) bg.template tick<TB + 1>();
        PTY_F8(1) bg.template tick<TB + 2>();
        PTY_F8(2) bg.template tick<TB + 3>();
        PTY_F8(3)
#undef PTY_F8
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = o[k];
    }
}

// twiddle table (forward sign), filled once per CTA: twg[g][i][q] = W128^(q (8 g + i))
PTY_DEV void f128_fill_twiddles(const Cta128& c) {
    for (int j = c.tid; j < 128; j += F128::NT) {
        float s, co;
        const int gi = j >> 2, qq = j & 3;        // gi = 8 g + i
        sincospi_f(2.0f * (float)(qq * gi) / 128.0f, &s, &co);
        c.twg[j] = make_float2(co, -s);
    }
}

// ------------------------------------------------------------------------------ TMEM exchange (T)
// out[8 g2 + i] = (value in[8 g + i] of the thread (g2, c)),  g = this thread's group.
// WAR: the partners' reads of the previous exchange must be complete before this thread overwrites
// its block; pass true unless a CTA barrier has been crossed since the previous exchange.
PTY_DEV void subpartition_sync(int tid) {      // the 4 warps {w, w+4, w+8, w+12} of one SM sub-partition
    asm volatile("bar.sync %0, 128;" ::"r"(1 + ((tid >> 5) & 3)) : "memory");
}
// FREE: also wait, after the reads, until the partners have read this thread's block, so that the block
// can be reused as a staging buffer (the next exchange then needs no WAR wait).
template <bool WAR, bool FREE> PTY_DEV void f128_tmem_exchange(const Cta128& c, float2 (&v)[32]) {
    if (WAR) {
        tmem_fence_before_sync();
        subpartition_sync(c.tid);
        tmem_fence_after_sync();
    }
    const unsigned mine = c.tm_x();
#pragma unroll
    for (int h = 0; h < 4; ++h) tmem_st8(mine + 16 * h, v, 8 * h);
    tmem_wait_st();
    tmem_fence_before_sync();
    subpartition_sync(c.tid);
    tmem_fence_after_sync();
    const unsigned col = 16u * (unsigned)c.g();
#pragma unroll
    for (int g2 = 0; g2 < 4; ++g2) tmem_ld8(c.tmq + 128u * g2 + col, v, 8 * g2);
    tmem_wait_ld();
    if (FREE) {
        tmem_fence_before_sync();
        subpartition_sync(c.tid);
        tmem_fence_after_sync();
    }
}

// ------------------------------------------------------------------------------ radix-4 stage (c)
// forward: v[8 q + i] -> twiddle W128^(q (8 g + i)) -> radix-4 over q -> v[8 k2 + i]
template <int T0, int T1, class BG> PTY_DEV void f128_radix4_fwd(const Cta128& c, float2 (&v)[32], BG& bg) {
    const float4* tw = reinterpret_cast<const float4*>(c.twg + 32 * c.g());
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float4 t01 = tw[2 * i], t23 = tw[2 * i + 1];
        float2 a0 = v[i];
        float2 a1 = cmul(v[8 + i], make_float2(t01.z, t01.w));
        float2 a2 = cmul(v[16 + i], make_float2(t23.x, t23.y));
        float2 a3 = cmul(v[24 + i], make_float2(t23.z, t23.w));
        bfly4<-1>(a0, a1, a2, a3);
        v[i] = a0; v[8 + i] = a1; v[16 + i] = a2; v[24 + i] = a3;
        if (i == 3) bg.template tick<T0>();
    }
    bg.template tick<T1>();
}
// inverse: v[8 k2 + i] -> inverse radix-4 over k2 -> conj twiddle -> v[8 q + i]
template <int T0, int T1, class BG> PTY_DEV void f128_radix4_inv(const Cta128& c, float2 (&v)[32], BG& bg) {
    const float4* tw = reinterpret_cast<const float4*>(c.twg + 32 * c.g());
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float4 t01 = tw[2 * i], t23 = tw[2 * i + 1];
        float2 a0 = v[i], a1 = v[8 + i], a2 = v[16 + i], a3 = v[24 + i];
        bfly4<+1>(a0, a1, a2, a3);
        v[i] = a0;
        v[8 + i] = cmulc(make_float2(t01.z, t01.w), a1);
        v[16 + i] = cmulc(make_float2(t23.x, t23.y), a2);
        v[24 + i] = cmulc(make_float2(t23.z, t23.w), a3);
        if (i == 3) bg.template tick<T0>();
    }
    bg.template tick<T1>();
}

// ------------------------------------------------------------------------------ forward, R -> K
// in: v[n1] = a[4 n1 + q][x];  out: v[8 k2 + i] = A[ky = c][kx = 8 g + i + 32 k2]  (unscaled).
// WAR0: the first exchange must wait for the partners' reads of the previous exchange (false when the
// preceding inverse ended with a FREE exchange).  14 ticks.
template <bool WAR0, class BG> PTY_DEV void f128_forward(const Cta128& c, float2 (&v)[32], BG& bg) {
    constexpr int P = F128::P;
    const int g = c.g(), cc = c.cc();
    // y axis
    bg.template tick<0>();
    fft32<-1, 1>(v, bg);
    f128_tmem_exchange<WAR0, false>(c, v);
    f128_radix4_fwd<5, 6>(c, v, bg);
    {   // S: thread (g, x = cc) holds ky = 8 g + i + 32 k2 in v[8 k2 + i]
        float2* s = c.X + (8 * g) * P + cc;
#pragma unroll
        for (int r = 0; r < 32; ++r) s[((r & 7) + 32 * (r >> 3)) * P] = v[r];
    }
    pty_cta_sync();
    {   // thread (xq = g, ky = cc) takes x = 4 n1x + xq
        const float2* s = c.X + cc * P + g;
#pragma unroll
        for (int n2 = 0; n2 < 8; ++n2) {     // in the order the first butterflies consume them
            v[n2] = s[4 * n2];
            v[8 + n2] = s[4 * (8 + n2)];
            v[16 + n2] = s[4 * (16 + n2)];
            v[24 + n2] = s[4 * (24 + n2)];
        }
    }
    // x axis
    bg.template tick<7>();
    fft32<-1, 8>(v, bg);
    f128_tmem_exchange<false, false>(c, v);
    f128_radix4_fwd<12, 13>(c, v, bg);
}

// ------------------------------------------------------------------------------ inverse, K -> R
// in: v[8 k2 + i] = A[ky = c][kx = 8 g + i + 32 k2];  out: v[n1] = a[4 n1 + q][x]  (unscaled: x N^2).
template <bool FREE, class BG, class BG2> PTY_DEV void f128_inverse(const Cta128& c, float2 (&v)[32], BG& bg, BG2& bg2) {
    constexpr int P = F128::P;
    const int g = c.g(), cc = c.cc();
    // x axis
    f128_radix4_inv<0, 1>(c, v, bg);
    f128_tmem_exchange<true, false>(c, v);
    fft32<+1, 2>(v, bg);
    bg.template tick<6>();
    {   // S: thread (xq = g, ky = cc) holds x = 4 n1x + xq in v[n1x]
        float2* s = c.X + cc * P + g;
#pragma unroll
        for (int n = 0; n < 32; ++n) s[4 * n] = v[n];
    }
    pty_cta_sync();
    {   // thread (g, x = cc) takes ky = 8 g + i + 32 k2 into v[8 k2 + i]
        const float2* s = c.X + (8 * g) * P + cc;
#pragma unroll
        for (int i = 0; i < 8; ++i) {        // in the order the butterflies consume them
            v[i] = s[i * P];
            v[8 + i] = s[(i + 32) * P];
            v[16 + i] = s[(i + 64) * P];
            v[24 + i] = s[(i + 96) * P];
        }
    }
    // y axis
    f128_radix4_inv<7, 8>(c, v, bg);
    f128_tmem_exchange<false, FREE>(c, v);
    bg2.template tick<0>();
    fft32<+1, 1>(v, bg2);
    bg2.template tick<5>();
}

PTY_DEV void f128_forward(const Cta128& c, float2 (&v)[32]) { NoBg bg; f128_forward<true>(c, v, bg); }
PTY_DEV void f128_inverse(const Cta128& c, float2 (&v)[32]) { NoBg bg, bg2; f128_inverse<false>(c, v, bg, bg2); }

}  // namespace pty
