// pty_fft128.cuh -- register-resident 128 x 128 2-D FFT for one CTA of 512 threads, in-place exchange.
//
// The whole wave lives in registers (32 complex values per thread); shared memory is only the
// exchange space between register phases.  A forward transform runs three phases (decimation in
// time), its inverse runs the exact mirror (decimation in frequency), so that
//   * the forward ENDS and the inverse STARTS in the same register layout ("L3", k space), and
//   * the inverse ENDS and the forward STARTS in the same layout ("L1", real space).
// A chain  ... F^-1 -> (pointwise in L1) -> F -> (pointwise in L3) -> F^-1 ...  therefore needs only
// TWO shared-memory exchanges per 2-D FFT, and every pointwise step of the method (object multiply,
// propagator, seeds, gradient products) is done on registers.
//
// IN-PLACE EXCHANGE.  Every element has ONE home slot in the exchange array X[128][P]:
//     slot(rho, c) = rho * P + 17 (c >> 4) + (c & 15),        P = 136 float2
// where (rho, c) = (4 k1y + q, x) between phases 1 and 2 and (4 k1y + k2y, 16 k1x + n2x) between
// phases 2 and 3.  In each phase a thread reads its 32 slots, transforms, and writes its results
// back to THE SAME 32 slots, so a slot is never touched by two threads between two barriers: one
// CTA barrier per exchange (two per 2-D FFT) is enough, no barrier separates a phase's loads from
// its stores, and the loads of a phase can be consumed as they arrive.
//
// Index split:  y = 4 n1 + q      (n1 < 32, q < 4)        ky = k1y + 32 k2y   (k1y < 32, k2y < 4)
//               x = 16 n1x + n2x  (n1x < 8, n2x < 16)     kx = k1x + 8 k2x    (k1x < 8,  k2x < 16)
//
//   L1: thread (q = tid >> 7, x = tid & 127)      holds a[y = 4 n1 + q][x],             n1 = 0..31
//   L2: thread (k1y = tid >> 4, n2x = tid & 15)   holds (q | k2y) x (n1x | k1x),        4 x 8
//   L3: thread (k1x = tid & 7, kyl = tid >> 3)    holds rows rho = kyl + 64 j, j < 2, i.e.
//        A[ky = (kyl >> 2) + 16 j + 32 (kyl & 3)][kx = k1x + 8 k2x],  k2x < 16,  register 16 j + k2x
//
//   forward:  radix-32 over n1 | X | twiddle W128^(q k1y), radix-4 over q, radix-8 over n1x,
//             twiddle W128^(n2x k1x) | X | radix-16 over n2x.
//   inverse:  the same steps conjugated, in reverse order.  Both are unscaled.
//
// Bank conflicts (8-byte accesses, one half-warp per wavefront): phase 1 touches 16 consecutive
// float2 of one row; phase 2 the same; phase 3 touches 8 slots at stride 17 in each of two rows
// whose offset P = 136 = 8 (mod 16) float2 -> all conflict-free.
#pragma once
#include "pty_fft.cuh"

namespace pty {

struct F128 {
    static constexpr int N = 128, NT = 512;
    static constexpr int P = 136;              // pitch of X (float2): 8 * 17
    static constexpr size_t xch_bytes = size_t(128) * P * sizeof(float2);
    // tables: twy[32][4], twx[8][16], Ey, Ex, My, Mx [128 each], red[64], tensor-memory base
    static constexpr size_t table_bytes = (128 + 128 + 4 * 128) * sizeof(float2) + 64 * sizeof(float) + 16;
    static constexpr size_t smem_bytes = xch_bytes + table_bytes;
};

struct Cta128 {
    int tid;
    float2* X;                       // exchange space
    float2 *twy, *twx;               // W128^(q k1y) [32][4];  W128^(n2x k1x) [8][16]   (forward sign)
    float2 *Ey, *Ex, *My, *Mx;       // [128] shift and propagator factors (Ex carries 1/N, Mx 1/N^2)
    float* red;
    unsigned tm;                     // tensor-memory address of this thread's 128-column staging block
    // L1 coordinates
    PTY_DEV int q() const { return tid >> 7; }
    PTY_DEV int x() const { return tid & 127; }
    // L3 coordinates
    PTY_DEV int k1x() const { return tid & 7; }
    PTY_DEV int kyl() const { return tid >> 3; }
    PTY_DEV int ky(int j) const { const int l = tid >> 3; return (l >> 2) + 16 * j + 32 * (l & 3); }
    // home slots
    PTY_DEV float2* slot1() const { return X + (tid >> 7) * F128::P + 17 * ((tid & 127) >> 4) + (tid & 15); }   // + 4 k P
    PTY_DEV float2* slot2() const { return X + 4 * (tid >> 4) * F128::P + (tid & 15); }                         // + q P + 17 n1x
    PTY_DEV float2* slot3() const { return X + (tid >> 3) * F128::P + 17 * (tid & 7); }                         // + 64 j P + n2
};

// cos / sin of 2 pi j / 32
PTY_DEV constexpr float c32(int j) {
    constexpr float t[9] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                            0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                            0.19509032201612826785f, 0.0f};
    j &= 31;
    return j <= 8 ? t[j] : j <= 16 ? -t[16 - j] : j <= 24 ? -t[j - 16] : t[32 - j];
}
PTY_DEV constexpr float s32(int j) { return c32(j - 8); }

template <int J, int DIR> PTY_DEV float2 mul_w32(float2 a) {
    constexpr float c = c32(J), s = s32(J);
    if constexpr (J % 32 == 0) return a;
    else if constexpr (J % 32 == 8) return mul_qi<DIR>(a);
    else return mul_cs<DIR>(a, c, s);
}

// 32-point DFT in registers, natural order in and out.  n = 8 n1 + n2, k = k1 + 4 k2.
template <int DIR> PTY_DEV void fft32(float2 (&v)[32]) {
#pragma unroll
    for (int n2 = 0; n2 < 8; ++n2) bfly4<DIR>(v[n2], v[8 + n2], v[16 + n2], v[24 + n2]);   // -> v[8 k1 + n2]
#define PTY_TW(K1, N2) v[8 * K1 + N2] = mul_w32<K1 * N2, DIR>(v[8 * K1 + N2]);
    PTY_TW(1, 1) PTY_TW(1, 2) PTY_TW(1, 3) PTY_TW(1, 4) PTY_TW(1, 5) PTY_TW(1, 6) PTY_TW(1, 7)
    PTY_TW(2, 1) PTY_TW(2, 2) PTY_TW(2, 3) PTY_TW(2, 4) PTY_TW(2, 5) PTY_TW(2, 6) PTY_TW(2, 7)
    PTY_TW(3, 1) PTY_TW(3, 2) PTY_TW(3, 3) PTY_TW(3, 4) PTY_TW(3, 5) PTY_TW(3, 6) PTY_TW(3, 7)
#undef PTY_TW
    float2 o[32];
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) {
        float2 w[8];
#pragma unroll
        for (int n2 = 0; n2 < 8; ++n2) w[n2] = v[8 * k1 + n2];
        RegFFT<8, DIR>::run(w);
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) o[k1 + 4 * k2] = w[k2];
    }
#pragma unroll
    for (int k = 0; k < 32; ++k) v[k] = o[k];
}

// twiddle tables (forward sign), filled once per CTA
PTY_DEV void f128_fill_twiddles(const Cta128& c) {
    for (int i = c.tid; i < 128; i += F128::NT) {
        float s, co;
        const int k1y = i >> 2, qq = i & 3;
        sincospi_f(2.0f * (float)(qq * k1y) / 128.0f, &s, &co);
        c.twy[i] = make_float2(co, -s);
        const int k1 = i >> 4, n2 = i & 15;
        sincospi_f(2.0f * (float)(k1 * n2) / 128.0f, &s, &co);
        c.twx[i] = make_float2(co, -s);
    }
}

// Background work interleaved with a transform: the transforms call bg.tick<K>() at 8 points spread
// evenly over their arithmetic (K = 0..7 in program order); the kernel bodies use the ticks to fetch
// the global data of the NEXT pointwise step in small chunks and park it in tensor memory.
struct NoBg { template <int K> PTY_DEV void tick() {} };

// a * w (DIR < 0) or a * conj(w) (DIR > 0), w a forward-sign twiddle
template <int DIR> PTY_DEV float2 mul_tw(float2 a, float2 w) { return DIR < 0 ? cmul(a, w) : cmulc(w, a); }

// ------------------------------------------------------------------------------ forward, L1 -> L3
// in: v[n1] = a[4 n1 + q][x];  out: v[16 j + k2x] = A[ky(j)][k1x + 8 k2x]  (unscaled).
// No barrier is needed before the first store: the slots written here were last read by this thread.
template <class BG> PTY_DEV void f128_forward(const Cta128& c, float2 (&v)[32], BG& bg) {
    constexpr int DIR = -1;
    constexpr int P = F128::P;
    {   // phase 1 (L1): radix-32 over n1, store to the home slots
        bg.template tick<0>();
        fft32<DIR>(v);
        bg.template tick<1>();
        float2* s1 = c.slot1();
#pragma unroll
        for (int k = 0; k < 32; ++k) s1[4 * k * P] = v[k];
    }
    pty_cta_sync();
    {   // phase 2 (L2): twiddle W128^(q k1y), radix-4 over q, radix-8 over n1x, twiddle W128^(n2x k1x)
        float2* s2 = c.slot2();
        const float2* ty = c.twy + 4 * (c.tid >> 4);
        const float2 wy1 = ty[1], wy2 = ty[2], wy3 = ty[3];
#pragma unroll
        for (int n1x = 0; n1x < 8; ++n1x) {
            float2 a0 = s2[17 * n1x], a1 = s2[P + 17 * n1x], a2 = s2[2 * P + 17 * n1x], a3 = s2[3 * P + 17 * n1x];
            a1 = cmul(a1, wy1); a2 = cmul(a2, wy2); a3 = cmul(a3, wy3);
            bfly4<DIR>(a0, a1, a2, a3);
            v[n1x] = a0; v[8 + n1x] = a1; v[16 + n1x] = a2; v[24 + n1x] = a3;       // -> v[8 k2y + n1x]
            if (n1x == 3) bg.template tick<2>();
        }
        bg.template tick<3>();
        const float2* tx = c.twx + (c.tid & 15);
#pragma unroll
        for (int k2y = 0; k2y < 4; ++k2y) {
            float2 w[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) w[i] = v[8 * k2y + i];
            RegFFT<8, DIR>::run(w);
            s2[k2y * P] = w[0];
#pragma unroll
            for (int k1 = 1; k1 < 8; ++k1) s2[k2y * P + 17 * k1] = cmul(w[k1], tx[16 * k1]);
            if (k2y == 1) bg.template tick<4>();
        }
        bg.template tick<5>();
    }
    pty_cta_sync();
    {   // phase 3 (L3): radix-16 over n2x
        const float2* s3 = c.slot3();
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            float2 w[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) w[i] = s3[64 * j * P + i];
            RegFFT<16, DIR>::run(w);
#pragma unroll
            for (int i = 0; i < 16; ++i) v[16 * j + i] = w[i];
            if (j == 0) bg.template tick<6>(); else bg.template tick<7>();
        }
    }
}
PTY_DEV void f128_forward(const Cta128& c, float2 (&v)[32]) { NoBg bg; f128_forward(c, v, bg); }

// ------------------------------------------------------------------------------ inverse, L3 -> L1
// in: v[16 j + k2x] = A[ky(j)][k1x + 8 k2x];  out: v[n1] = a[4 n1 + q][x]  (unscaled: x N^2).
// MY: 0 none, +1 multiply the spectrum by My[ky], -1 by conj(My[ky]) (the k_y factor of the
// propagator, applied where every thread sees only 4 distinct ky).
template <int MY, class BG> PTY_DEV void f128_inverse(const Cta128& c, float2 (&v)[32], BG& bg) {
    constexpr int DIR = +1;
    constexpr int P = F128::P;
    {   // phase 3' (L3): inverse radix-16 over k2x, store to the home slots
        float2* s3 = c.slot3();
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            float2 w[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) w[i] = v[16 * j + i];
            RegFFT<16, DIR>::run(w);
#pragma unroll
            for (int i = 0; i < 16; ++i) s3[64 * j * P + i] = w[i];
            if (j == 0) bg.template tick<0>(); else bg.template tick<1>();
        }
    }
    pty_cta_sync();
    {   // phase 2' (L2): conj twiddle, inverse radix-8 over k1x, (My), inverse radix-4 over k2y, conj twiddle
        float2* s2 = c.slot2();
        const int k1y = c.tid >> 4;
        const float2* tx = c.twx + (c.tid & 15);
#pragma unroll
        for (int k2y = 0; k2y < 4; ++k2y) {
            float2 w[8];
            w[0] = s2[k2y * P];
#pragma unroll
            for (int k1 = 1; k1 < 8; ++k1) w[k1] = cmulc(tx[16 * k1], s2[k2y * P + 17 * k1]);
            RegFFT<8, DIR>::run(w);
            if (MY != 0) {
                float2 m = c.My[k1y + 32 * k2y];
                if (MY < 0) m.y = -m.y;
#pragma unroll
                for (int i = 0; i < 8; ++i) w[i] = cmul(w[i], m);
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) v[8 * k2y + i] = w[i];
            if (k2y == 1) bg.template tick<2>();
        }
        bg.template tick<3>();
        const float2* ty = c.twy + 4 * k1y;
        const float2 wy1 = ty[1], wy2 = ty[2], wy3 = ty[3];
#pragma unroll
        for (int n1x = 0; n1x < 8; ++n1x) {
            float2 a0 = v[n1x], a1 = v[8 + n1x], a2 = v[16 + n1x], a3 = v[24 + n1x];
            bfly4<DIR>(a0, a1, a2, a3);                                              // -> q = 0..3
            s2[17 * n1x] = a0;
            s2[P + 17 * n1x] = cmulc(wy1, a1);
            s2[2 * P + 17 * n1x] = cmulc(wy2, a2);
            s2[3 * P + 17 * n1x] = cmulc(wy3, a3);
            if (n1x == 3) bg.template tick<4>();
        }
        bg.template tick<5>();
    }
    pty_cta_sync();
    {   // phase 1' (L1): inverse radix-32 over k1y
        const float2* s1 = c.slot1();
#pragma unroll
        for (int n2 = 0; n2 < 8; ++n2) {         // in the order the first butterflies consume them
            v[n2] = s1[4 * n2 * P];
            v[8 + n2] = s1[4 * (8 + n2) * P];
            v[16 + n2] = s1[4 * (16 + n2) * P];
            v[24 + n2] = s1[4 * (24 + n2) * P];
        }
        bg.template tick<6>();
        fft32<DIR>(v);
        bg.template tick<7>();
    }
}
template <int MY> PTY_DEV void f128_inverse(const Cta128& c, float2 (&v)[32]) { NoBg bg; f128_inverse<MY>(c, v, bg); }

}  // namespace pty
