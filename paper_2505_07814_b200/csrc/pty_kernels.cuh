// pty_kernels.cuh -- bodies of the forward and adjoint kernels (one CTA, or one 4-CTA cluster
// for N = 256, per (position b, probe mode m)); the pointwise work of the method is fused into
// the first register stage ("stage A") of the FFT pass that follows it.
//
// Orientation: after every 2-D FFT (two passes) the wave in shared memory is S[row = y][line = x]
// (or [k_y][k_x]); every fused operation below happens in that orientation, where global-memory
// accesses are contiguous along the line index = lanes of a warp.
//
// Scaling: passes are unscaled.  The unitary factors are folded into the tables:
//   Ex carries 1/N  (probe shift F^-1, and the final F of the adjoint),
//   Mx carries 1/N^2 (F^-1 M F of a propagation and of its adjoint),
//   the far field and the seed carry 1/N explicitly.
//
// Paper references: PAPER.md:75-90 (crop, shift, Eq. 3 multislice, Eq. 4 propagator), :66-71 (Eq. 2
// mode sum), :126-131 (Eq. 5); adjoint steps B1-B8 as derived in DESIGN.md "Adjoint".
#pragma once
#include "pty_fft.cuh"

namespace pty {

struct KArgs {
    int Nz, H, W, M, B;
    int Nobj, MT;         // object states (Eq. 2) and MT = M * Nobj items per position:
                          // item = b MT + n M + m runs probe mode m through object state n
    int tilt_mode;        // 0 none, 1 global, 2 per position
    int save_hat;         // keep propagated spectra (tilt / dz gradients)
    float dz, lambda, dx;
    const float2* object;      // [Nobj][Nz][H][W]
    const float2* probe_hat;   // [M][N][N]  unitary spectrum of the probe
    const float* positions;    // [B][2]
    const float* tilt;         // [2] or [B][2] or null
    const float* meas;         // [B][N][N]
    const float2* prop_y;      // [N] exp(i chi_y) (tilt_mode 0/1)
    const float2* prop_x;      // [N] exp(i chi_x)
    float* I;                  // [B][N][N]   mode-summed intensity
    float2* ws_psi;            // [B][M][Nz][N][N]  wave incident on every slice
    float2* ws_Psi;            // [B][M][N][N]      far field (unitary)
    float2* ws_hat;            // [B][M][Nz-1][N][N] spectrum of psi_{s+1} (times 1/N), optional
    float2* GP_hat;            // [M][N][N]   sum_b conj(E_b) F[g_psi0]
    float* dsum;               // [B][4]      sum_k D (k_py, k_px, |k_p|^2)
    float* seed_w;             // [B][N][N] seed weights 2 (dL/dI) / N: thread order [r][tid] for N = 128, else natural
    int* flags;                // sticky device flags (bit 0: a crop was clamped)
    float2* g_object;          // [Nobj][Nz][H][W]
    float* g_pos;              // [B][2]
};

// item -> position b, probe mode m, offset of object state n in `object` / `g_object`
PTY_DEV void decode_item(const KArgs& A, int item, int& b, int& m, size_t& obj_off) {
    b = item / A.MT;
    const int mm = item - b * A.MT;
    const int n = mm / A.M;
    m = mm - n * A.M;
    obj_off = (size_t)n * A.Nz * A.H * A.W;
}

template <int N> PTY_DEV float kp_of(int j) { return (float)(j < N / 2 ? j : j - N) * (1.0f / N); }

// --------------------------------------------------------------------------- per-CTA set-up (a1)
// F1: r = floor(p + 0.5), Delta = p - r; tables: twiddles, shift factors E (F2), propagator (F4).
template <int N, int NT>
PTY_DEV void setup_factors(int tid, float2* Ey, float2* Ex, float2* My, float2* Mx, float* red, const KArgs& A,
                           int b, int& ry, int& rx) {
    const double py = (double)A.positions[2 * b], px = (double)A.positions[2 * b + 1];
    const double fy = floor(py + 0.5), fx = floor(px + 0.5);
    const float dy = (float)(py - fy), dxp = (float)(px - fx);
    int iy = (int)fy, ix = (int)fx;
    const int cy = min(max(iy, 0), A.H - N), cx = min(max(ix, 0), A.W - N);
    if ((cy != iy || cx != ix) && tid == 0) flag_or(A.flags, 1);
    ry = cy; rx = cx;
    double ty = 0.0, tx = 0.0;
    if (A.tilt_mode == 2) { ty = (double)A.tilt[2 * b]; tx = (double)A.tilt[2 * b + 1]; }
    for (int j = tid; j < N; j += NT) {
        float s, co;
        const float kp = kp_of<N>(j);
        sincospi_f(-2.0f * kp * dy, &s, &co);
        Ey[j] = make_float2(co, s);
        sincospi_f(-2.0f * kp * dxp, &s, &co);
        Ex[j] = make_float2(co * (1.0f / N), s * (1.0f / N));
        float2 my, mx;
        if (A.tilt_mode == 2) {
            const double k = (double)kp / (double)A.dx;
            const double quad = -3.14159265358979323846 * (double)A.lambda * (double)A.dz * k * k;
            const double lin = 2.0 * 3.14159265358979323846 * (double)A.dz * k;
            const double chy = quad + lin * tan(ty), chx = quad + lin * tan(tx);
            my = make_float2((float)cos(chy), (float)sin(chy));
            mx = make_float2((float)cos(chx), (float)sin(chx));
        } else {
            my = A.prop_y[j];
            mx = A.prop_x[j];
        }
        My[j] = my;
        Mx[j] = make_float2(mx.x * (1.0f / (N * N)), mx.y * (1.0f / (N * N)));
    }
    if (tid < 64) red[tid] = 0.f;
}

template <class SH>
PTY_DEV void setup_tables(const Cta<SH>& c, const KArgs& A, int b, int& ry, int& rx) {
    constexpr int N = SH::N;
    setup_factors<N, SH::NT>(c.tid, c.Ey, c.Ex, c.My, c.Mx, c.red, A, b, ry, rx);
    for (int j = c.tid; j < N; j += SH::NT) {
        float s, co;
        sincospi_f(2.0f * (float)j / (float)N, &s, &co);
        c.tw[j] = make_float2(co, -s);
    }
    pty_cta_sync();
}

// --------------------------------------------------------------------------- stage-A inputs
// K-space steps see the wave TRANSPOSED (pty_fft.cuh, fft_2d): row = k_x, line = k_y; every k-space workspace array
// of this kernel family is stored in that order, [k_x][k_y].
// a2: E_b . P^ (k space), source = global memory
struct InProbe {
    const float2* Ph;
    template <class SH, int R>
    PTY_DEV void load(const Cta<SH>& c, int n2, int, int gline, float2 (&v)[R]) {
        using I = ShapeInfo<SH>;
        const float2 eyl = c.Ey[gline];
#pragma unroll
        for (int n1 = 0; n1 < R; ++n1) {
            const int row = I::R2 * n1 + n2;
            v[n1] = cmul(cmul(ldg2(Ph + row * I::N + gline), c.Ex[row]), eyl);
        }
    }
};

// a3 + a4: save psi_{s-1}, gather the object patch, phi_s = O_b[s] . psi_{s-1}
struct InFwdObj {
    const float2* obj;   // object + s*H*W + ry*W + rx
    int W;
    float2* save;        // ws_psi[b][m][s]
    // v[n1] = psi_{s-1}(row R2 n1 + n2, line) on entry (fused step, pty_fft.cuh stage_b_op_a), phi_s on return
    template <class SH, int R>
    PTY_DEV void apply(const Cta<SH>&, int n2, int, int gline, float2 (&v)[R]) {
        using I = ShapeInfo<SH>;
        float2 o[R];
#pragma unroll
        for (int n1 = 0; n1 < R; ++n1) o[n1] = ldg2(obj + (size_t)(I::R2 * n1 + n2) * W + gline);
#pragma unroll
        for (int n1 = 0; n1 < R; ++n1) {
            const int row = I::R2 * n1 + n2;
            st_stream2(save + row * I::N + gline, v[n1]);
            v[n1] = cmul(v[n1], o[n1]);
        }
    }
};

// a4: multiply the spectrum by the propagator M = Mx[row] My[line] (/N^2); optionally keep it
struct InFwdProp {
    float2* save;   // ws_hat[b][m][s] or null
    template <class SH, int R>
    PTY_DEV void apply(const Cta<SH>& c, int n2, int, int gline, float2 (&v)[R]) {
        using I = ShapeInfo<SH>;
        const float2 myl = c.My[gline];
#pragma unroll
        for (int n1 = 0; n1 < R; ++n1) {
            const int row = I::R2 * n1 + n2;
            const float2 w = cmul(v[n1], cmul(c.Mx[row], myl));
            if (save) st_stream2(save + row * I::N + gline, w);
            v[n1] = w;
        }
    }
};

// a7 (B1): g_Psi = w Psi with the seed weights w = 2 (dL/dI) / N written by the loss kernels (pty_pointwise.cuh;
// plain sum: dL/dI = 1 - a / sqrt(I), zero where I = 0); the 1/N is that of the F^-1 (B2)
struct InSeed {
    const float2* Psi;
    const float* Wt;
    template <class SH, int R>
    PTY_DEV void load(const Cta<SH>&, int n2, int, int gline, float2 (&v)[R]) {
        using SI = ShapeInfo<SH>;
        float wv[R];
#pragma unroll
        for (int n1 = 0; n1 < R; ++n1) {
            const int idx = (SI::R2 * n1 + n2) * SI::N + gline;
            v[n1] = ld_stream2(Psi + idx);
            wv[n1] = ldg1(Wt + idx);
        }
#pragma unroll
        for (int n1 = 0; n1 < R; ++n1) v[n1] = cscale(v[n1], wv[n1]);
    }
};

// a9/a10 (B3, B4): g_object patch += conj(psi_{s-1}) g;  g <- conj(O_b[s]) g
struct InBwdObj {
    const float2* obj;
    int W;
    const float2* psi;   // ws_psi[b][m][s]
    float2* gobj;        // g_object + s*H*W + ry*W + rx
    template <class SH, int R>
    PTY_DEV void apply(const Cta<SH>&, int n2, int, int gline, float2 (&v)[R]) {
        using I = ShapeInfo<SH>;
        constexpr int CH = 8;
#pragma unroll
        for (int h = 0; h < R; h += CH) {
            float2 ps[CH], o[CH];
#pragma unroll
            for (int q = 0; q < CH; ++q) {
                const int row = I::R2 * (h + q) + n2;
                ps[q] = ld_stream2(psi + row * I::N + gline);
                o[q] = ldg2(obj + (size_t)row * W + gline);
            }
#pragma unroll
            for (int q = 0; q < CH; ++q) {
                const int row = I::R2 * (h + q) + n2;
                const float2 g = v[h + q];
                red_add2(gobj + (size_t)row * W + gline, cmulc(ps[q], g));
                v[h + q] = cmulc(o[q], g);
            }
        }
    }
};

// a9 (B5) + a13 (B8): D-sums against the kept spectrum, then multiply by conj(M) (/N^2)
struct InBwdProp {
    const float2* hat;   // ws_hat[b][m][s-1] or null
    float acc_ky, acc_kx, acc_k2;
    template <class SH, int R>
    PTY_DEV void apply(const Cta<SH>& c, int n2, int, int gline, float2 (&v)[R]) {
        using I = ShapeInfo<SH>;
        const float2 myl = c.My[gline];
        const float kyl = kp_of<I::N>(gline);
#pragma unroll
        for (int n1 = 0; n1 < R; ++n1) {
            const int row = I::R2 * n1 + n2;
            const float2 g = v[n1];
            if (hat) {
                const float2 hs = ld_stream2(hat + row * I::N + gline);
                const float d = hs.x * g.y - hs.y * g.x;       // Im(conj(psi^) g^)
                const float kxr = kp_of<I::N>(row);
                acc_ky += d * kyl;
                acc_kx += d * kxr;
                acc_k2 += d * (kyl * kyl + kxr * kxr);
            }
            v[n1] = cmulc(cmul(c.Mx[row], myl), g);
        }
    }
};

// plain global source (probe spectrum prep, probe-gradient finalisation)
struct InGlobal {
    const float2* src;
    template <class SH, int R>
    PTY_DEV void load(const Cta<SH>&, int n2, int, int gline, float2 (&v)[R]) {
        using I = ShapeInfo<SH>;
#pragma unroll
        for (int n1 = 0; n1 < R; ++n1) v[n1] = ldg2(src + (I::R2 * n1 + n2) * I::N + gline);
    }
};

// --------------------------------------------------------------------------- block reductions
template <class SH>
PTY_DEV void block_accumulate(const Cta<SH>& c, int slot, float v) {
    v = warp_sum(v);
    if (warp_leader()) red_add_shared(c.red + slot, v);
}

// --------------------------------------------------------------------------- forward (a2-a5)
template <class SH>
PTY_DEV void fwd_body(const KArgs& A, const Cta<SH>& c, int item) {
    using I = ShapeInfo<SH>;
    constexpr int N = SH::N;
    int b, m;
    size_t obj_off;
    decode_item(A, item, b, m, obj_off);
    int ry, rx;
    setup_tables(c, A, b, ry, rx);
    const size_t NN = (size_t)N * N;
    const size_t bm = (size_t)item;
    {   // psi_0 = F^-1[E . P^] (up to the last stage B: the object multiply of slice 0 is fused into it)
        InProbe in{A.probe_hat + (size_t)m * NN};
        fft_begin<SH, +1>(c, in);
    }
    for (int s = 0; s < A.Nz; ++s) {
        InFwdObj in{A.object + obj_off + ((size_t)s * A.H + ry) * A.W + rx, A.W, A.ws_psi + (bm * A.Nz + s) * NN};
        fft_link<SH, +1, -1>(c, in);
        if (s == A.Nz - 1) break;
        InFwdProp ip{A.save_hat ? A.ws_hat + (bm * (A.Nz - 1) + s) * NN : nullptr};
        fft_link<SH, -1, +1>(c, ip);
    }
    fft_end<SH, -1>(c);
    // a5: Psi = F[phi_Nz] (unitary), I += |Psi|^2; both in the transposed k-space order [k_x][k_y]
    float2* Psi = A.ws_Psi + bm * NN;
    float* Ib = A.I + (size_t)b * NN;
#pragma unroll 4
    for (int it = 0; it < I::SWEEP; ++it) {
        const int idx = it * I::NT + c.tid;
        const int row = idx / I::NL, line = idx % I::NL, gline = c.rank * I::NL + line;
        const float2 v = cscale(c.S[row * I::PITCH + line], 1.0f / N);
        st_stream2(Psi + row * N + gline, v);
        red_add(Ib + row * N + gline, v.x * v.x + v.y * v.y);
    }
}

// --------------------------------------------------------------------------- adjoint (a7-a13)
template <class SH>
PTY_DEV void bwd_body(const KArgs& A, const Cta<SH>& c, int item) {
    using I = ShapeInfo<SH>;
    constexpr int N = SH::N;
    int b, m;
    size_t obj_off;
    decode_item(A, item, b, m, obj_off);
    int ry, rx;
    setup_tables(c, A, b, ry, rx);
    const size_t NN = (size_t)N * N;
    const size_t bm = (size_t)item;
    {   // B1, B2
        InSeed in{A.ws_Psi + bm * NN, A.seed_w + (size_t)b * NN};
        fft_begin<SH, +1>(c, in);
    }
    InBwdProp ip{nullptr, 0.f, 0.f, 0.f};
    for (int s = A.Nz - 1; s >= 0; --s) {
        const size_t off = obj_off + ((size_t)s * A.H + ry) * A.W + rx;
        InBwdObj in{A.object + off, A.W, A.ws_psi + (bm * A.Nz + s) * NN, A.g_object + off};
        fft_link<SH, +1, -1>(c, in);
        if (s == 0) break;
        ip.hat = A.save_hat ? A.ws_hat + (bm * (A.Nz - 1) + (s - 1)) * NN : nullptr;
        fft_link<SH, -1, +1>(c, ip);
    }
    fft_end<SH, -1>(c);
    // B6, B7: g^_0 = F[g_psi0]; probe-gradient accumulation and the position gradient
    const float2* Ph = A.probe_hat + (size_t)m * NN;
    float2* GP = A.GP_hat + (size_t)m * NN;
    float accy = 0.f, accx = 0.f;
#pragma unroll 4
    for (int it = 0; it < I::SWEEP; ++it) {
        const int idx = it * I::NT + c.tid;
        const int row = idx / I::NL, line = idx % I::NL, gline = c.rank * I::NL + line;
        const float2 g = c.S[row * I::PITCH + line];
        const float2 e = cmul(c.Ex[row], c.Ey[gline]);           // E / N (row = k_x, line = k_y)
        red_add2(GP + row * N + gline, cmulc(e, g));
        const float2 ep = cmul(e, ldg2(Ph + row * N + gline));
        const float t = g.x * ep.y - g.y * ep.x;                 // Im(conj(g^_0) E P^)
        accy += kp_of<N>(gline) * t;
        accx += kp_of<N>(row) * t;
    }
    block_accumulate(c, 0, accy);
    block_accumulate(c, 1, accx);
    if (A.save_hat) {
        block_accumulate(c, 2, ip.acc_ky);
        block_accumulate(c, 3, ip.acc_kx);
        block_accumulate(c, 4, ip.acc_k2);
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

// --------------------------------------------------------------------------- plain 2-D FFT of M planes
// dst = scale * F^{DIR}[src] (+ dst if accumulate); used for P^ = F[P] and g_probe = F^-1[G^_P].
template <class SH, int DIR>
PTY_DEV void fft2_body(const float2* src, float2* dst, float scale, int accumulate, const Cta<SH>& c, int item) {
    using I = ShapeInfo<SH>;
    constexpr int N = SH::N;
    for (int j = c.tid; j < N; j += SH::NT) {
        float s, co;
        sincospi_f(2.0f * (float)j / (float)N, &s, &co);
        c.tw[j] = make_float2(co, -s);
    }
    pty_cta_sync();
    const size_t NN = (size_t)N * N;
    InGlobal in{src + (size_t)item * NN};
    fft_2d<SH, DIR>(c, in);          // DIR < 0: natural [y][x] -> transposed [k_x][k_y]; DIR > 0: the reverse
    float2* out = dst + (size_t)item * NN;
    for (int it = 0; it < I::SWEEP; ++it) {
        const int idx = it * I::NT + c.tid;
        const int row = idx / I::NL, line = idx % I::NL, gline = c.rank * I::NL + line;
        float2 v = cscale(c.S[row * I::PITCH + line], scale);
        if (accumulate) v = cadd(v, out[row * N + gline]);
        out[row * N + gline] = v;
    }
}

}  // namespace pty
