// pty_fft128.cuh -- register-resident 128 x 128 2-D FFT for one CTA of 512 threads.
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
// Index split:  y = 4 n1 + q      (n1 < 32, q < 4)        ky = k1y + 32 k2y   (k1y < 32, k2y < 4)
//               x = 16 n1x + n2x  (n1x < 8, n2x < 16)     kx = k1x + 8 k2x    (k1x < 8,  k2x < 16)
//
//   L1: thread (q = tid >> 7, x = tid & 127)            holds a[y = 4 n1 + q][x],            n1  = 0..31
//   L2: thread (k1y = tid >> 4, n2x = tid & 15)         holds (q | k2y) x (n1x | k1x),       4 x 8
//   L3: thread (k1x = tid & 7, ky0 = tid >> 3)          holds A[ky0 + 64 j][k1x + 8 k2x],    j < 2, k2x < 16
//
//   forward:  radix-32 over n1, twiddle W128^(q k1y) | X1 | radix-4 over q, radix-8 over n1x,
//             twiddle W128^(n2x k1x) | X2 | radix-16 over n2x.
//   inverse:  the same steps conjugated, in reverse order.  Both are unscaled.
//
// Exchange X1 is the array E1[4 k1y + q][x] (pitch 128); X2 is E2[ky][17 k1x + n2x] (pitch 136):
// both sides of both exchanges touch 16 consecutive float2 per half-warp, or 8 lanes at stride 17
// in two rows whose offset is 16 banks -> conflict-free 8-byte accesses.
#pragma once
#include "pty_fft.cuh"

namespace pty {

struct F128 {
    static constexpr int N = 128, NT = 512;
    static constexpr int P1 = 128;             // pitch of E1 (float2)
    static constexpr int P2 = 136;             // pitch of E2 (float2): 8 * 17
    static constexpr size_t xch_bytes = size_t(128) * P2 * sizeof(float2);
    // tables: twy[4][32], twx[8][16], Ey, Ex, My, Mx [128 each], red[64]
    static constexpr size_t table_bytes = (128 + 128 + 4 * 128) * sizeof(float2) + 64 * sizeof(float);
    static constexpr size_t smem_bytes = xch_bytes + table_bytes;
};

struct Cta128 {
    int tid;
    float2* X;                       // exchange space
    float2 *twy, *twx;               // W128^(q k1y) [4][32];  W128^(n2x k1x) [8][16]   (forward sign)
    float2 *Ey, *Ex, *My, *Mx;       // [128] shift and propagator factors (Ex carries 1/N, Mx 1/N^2)
    float* red;
    // L1 coordinates
    PTY_DEV int q() const { return tid >> 7; }
    PTY_DEV int x() const { return tid & 127; }
    // L3 coordinates
    PTY_DEV int k1x() const { return tid & 7; }
    PTY_DEV int ky0() const { return tid >> 3; }
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
        const int qq = i >> 5, k1y = i & 31;
        sincospi_f(2.0f * (float)(qq * k1y) / 128.0f, &s, &co);
        c.twy[i] = make_float2(co, -s);
        const int k1 = i >> 4, n2 = i & 15;
        sincospi_f(2.0f * (float)(k1 * n2) / 128.0f, &s, &co);
        c.twx[i] = make_float2(co, -s);
    }
}

template <int DIR> PTY_DEV float2 tw_dir(float2 w) { return DIR < 0 ? w : make_float2(w.x, -w.y); }

// ------------------------------------------------------------------------------ forward, L1 -> L3
// in: v[n1] = a[4 n1 + q][x];  out: v[16 j + k2x] = A[ky0 + 64 j][k1x + 8 k2x]  (unscaled).
// The caller guarantees nobody is still reading the exchange space (a CTA barrier sits at the end
// of every transform).
PTY_DEV void f128_forward(const Cta128& c, float2 (&v)[32]) {
    constexpr int DIR = -1;
    {   // phase 1 (L1): radix-32 over n1, twiddle W128^(q k1y), write E1[4 k1y + q][x]
        fft32<DIR>(v);
        const int q = c.q(), x = c.x();
        if (q != 0) {
            const float2* tw = c.twy + 32 * q;
#pragma unroll
            for (int k = 1; k < 32; ++k) v[k] = cmul(v[k], tw[k]);
        }
#pragma unroll
        for (int k = 0; k < 32; ++k) c.X[(4 * k + q) * F128::P1 + x] = v[k];
    }
    pty_cta_sync();
    {   // phase 2 (L2): radix-4 over q, radix-8 over n1x, twiddle W128^(n2x k1x), write E2
        const int k1y = c.tid >> 4, n2x = c.tid & 15;
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
            for (int n1x = 0; n1x < 8; ++n1x) v[8 * q + n1x] = c.X[(4 * k1y + q) * F128::P1 + 16 * n1x + n2x];
        pty_cta_sync();
#pragma unroll
        for (int n1x = 0; n1x < 8; ++n1x) bfly4<DIR>(v[n1x], v[8 + n1x], v[16 + n1x], v[24 + n1x]);   // -> v[8 k2y + n1x]
        float2 tw[8];
#pragma unroll
        for (int k1 = 1; k1 < 8; ++k1) tw[k1] = c.twx[16 * k1 + n2x];
#pragma unroll
        for (int k2y = 0; k2y < 4; ++k2y) {
            float2 w[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) w[i] = v[8 * k2y + i];
            RegFFT<8, DIR>::run(w);
            float2* row = c.X + (k1y + 32 * k2y) * F128::P2 + n2x;
            row[0] = w[0];
#pragma unroll
            for (int k1 = 1; k1 < 8; ++k1) row[17 * k1] = cmul(w[k1], tw[k1]);
        }
    }
    pty_cta_sync();
    {   // phase 3 (L3): radix-16 over n2x
        const int k1x = c.k1x(), ky0 = c.ky0();
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int n2 = 0; n2 < 16; ++n2) v[16 * j + n2] = c.X[(ky0 + 64 * j) * F128::P2 + 17 * k1x + n2];
        pty_cta_sync();
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            float2 w[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) w[i] = v[16 * j + i];
            RegFFT<16, DIR>::run(w);
#pragma unroll
            for (int i = 0; i < 16; ++i) v[16 * j + i] = w[i];
        }
    }
}

// ------------------------------------------------------------------------------ inverse, L3 -> L1
// in: v[16 j + k2x] = A[ky0 + 64 j][k1x + 8 k2x];  out: v[n1] = a[4 n1 + q][x]  (unscaled: x N^2).
// MY: 0 none, +1 multiply the spectrum by My[ky], -1 by conj(My[ky]) (the k_y factor of the
// propagator, applied where every thread sees only 4 distinct ky).
template <int MY> PTY_DEV void f128_inverse(const Cta128& c, float2 (&v)[32]) {
    constexpr int DIR = +1;
    {   // phase 3' (L3): inverse radix-16 over k2x, write E2[ky][17 k1x + n2x]
        const int k1x = c.k1x(), ky0 = c.ky0();
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            float2 w[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) w[i] = v[16 * j + i];
            RegFFT<16, DIR>::run(w);
            float2* row = c.X + (ky0 + 64 * j) * F128::P2 + 17 * k1x;
#pragma unroll
            for (int i = 0; i < 16; ++i) row[i] = w[i];
        }
    }
    pty_cta_sync();
    {   // phase 2' (L2): conj twiddle, inverse radix-8 over k1x, (My), inverse radix-4 over k2y, write E1
        const int k1y = c.tid >> 4, n2x = c.tid & 15;
#pragma unroll
        for (int k2y = 0; k2y < 4; ++k2y)
#pragma unroll
            for (int k1 = 0; k1 < 8; ++k1) v[8 * k2y + k1] = c.X[(k1y + 32 * k2y) * F128::P2 + 17 * k1 + n2x];
        pty_cta_sync();
        float2 tw[8];
#pragma unroll
        for (int k1 = 1; k1 < 8; ++k1) tw[k1] = c.twx[16 * k1 + n2x];
#pragma unroll
        for (int k2y = 0; k2y < 4; ++k2y) {
            float2 w[8];
            w[0] = v[8 * k2y];
#pragma unroll
            for (int k1 = 1; k1 < 8; ++k1) w[k1] = cmulc(tw[k1], v[8 * k2y + k1]);
            RegFFT<8, DIR>::run(w);
            if (MY != 0) {
                float2 m = c.My[k1y + 32 * k2y];
                if (MY < 0) m.y = -m.y;
#pragma unroll
                for (int i = 0; i < 8; ++i) w[i] = cmul(w[i], m);
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) v[8 * k2y + i] = w[i];
        }
#pragma unroll
        for (int n1x = 0; n1x < 8; ++n1x) {
            bfly4<DIR>(v[n1x], v[8 + n1x], v[16 + n1x], v[24 + n1x]);   // -> v[8 q + n1x]
#pragma unroll
            for (int q = 0; q < 4; ++q) c.X[(4 * k1y + q) * F128::P1 + 16 * n1x + n2x] = v[8 * q + n1x];
        }
    }
    pty_cta_sync();
    {   // phase 1' (L1): conj twiddle W128^(-q k1y), inverse radix-32 over k1y
        const int q = c.q(), x = c.x();
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = c.X[(4 * k + q) * F128::P1 + x];
        pty_cta_sync();
        if (q != 0) {
            const float2* tw = c.twy + 32 * q;
#pragma unroll
            for (int k = 1; k < 32; ++k) v[k] = cmulc(tw[k], v[k]);
        }
        fft32<DIR>(v);
    }
}

}  // namespace pty
