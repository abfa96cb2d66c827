// pty_pointwise.cuh -- the HBM-bound pointwise / reduction kernels around the two big FFT kernels:
//   * the paper's loss family, Eq. 5-9: per-minibatch sums, the normalised terms and the seed
//     weights dL/dI that start the adjoint (pty_loss_sums_kernel, pty_loss_finalize_kernel, pty_seed_kernel);
//   * the amplitude / phase object parameterisation: O = A exp(i phi), its chain rule and the L1
//     sparsity term on the phase patches (Eq. 8);
//   * the per-iteration constraints of the paper's timed runs (PAPER.md:147, :289, :301-312 Eq. 13, :539):
//     probe-mode orthogonalisation, r_z depth blur, phase positivity, amplitude clamp.
// Readings R27-R31 of DESIGN.md apply.  Every kernel is a single pass over its arrays.
#pragma once
#include "pty_port.cuh"

namespace pty {

// workspace statistics (double), zeroed by the forward: sums over the minibatch, then terms and coefficients
enum : int { ST_S = 0, ST_A = 1, ST_A2 = 2, ST_P = 3, ST_SPARSE_SUM = 4, ST_LG = 8, ST_LP = 9, ST_LPB = 10, ST_LS = 11,
             ST_CG = 12, ST_CP = 13, ST_CPB = 14, ST_COUNT = 16 };

struct LossCfg {
    float w_gaussian, w_poisson, w_pacbed, w_sparse, eps;
};

PTY_DEV double block_sum_256(double v, double* part) {      // 256 threads; result valid in thread 0
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < 8; ++w) s += part[w];
    return s;
}

// Visits every detector pixel of one position once: f(I, a, w_index, natural_index).
// TORD (N = 128): I is in the forward kernel's thread order, pairs [r / 2][128 o + ky][r & 1]; the measured amplitudes
// (natural order) pass through a 32-row shared tile; w_index is the adjoint kernel's thread order [r][128 o + ky].
// Otherwise I and the seed weights are transposed, [k_x][k_y], and a is natural.  256 threads.
template <bool TORD, class F>
PTY_DEV void sweep_position(const float* __restrict__ Ib, const float* __restrict__ ab, int N, float (*tile)[129], F&& f) {
    const int t = threadIdx.x;
    if (TORD) {
        const float2* I2 = reinterpret_cast<const float2*>(Ib);
        for (int ky0 = 0; ky0 < 128; ky0 += 32) {
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const int idx = j * 256 + t, row = idx >> 7, kx = idx & 127;
                tile[row][kx] = __ldg(ab + (ky0 + row) * 128 + kx);
            }
            __syncthreads();
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int idx = j * 256 + t, row = idx & 31, kx = 2 * (idx >> 5);
                const int r = 8 * (kx >> 5) + (kx & 7), g = (kx >> 3) & 3, ky = ky0 + row;
                const float2 iv = __ldg(I2 + (r >> 1) * 512 + 128 * g + ky);
                f(iv.x, tile[row][kx], r * 512 + 128 * g + ky, ky * 128 + kx);
                f(iv.y, tile[row][kx + 1], (r + 1) * 512 + 128 * g + ky, ky * 128 + kx + 1);
            }
            __syncthreads();
        }
    } else {
        // N = 64 / 256: I and the seed weights are in the transposed k-space order [k_x][k_y] of the shared-memory-pass
        // kernels (pty_fft.cuh, fft_2d); the measured amplitudes are natural, [k_y][k_x]
        // A direct walk of the natural index: I is read and the weights are written at a stride of N floats (one sector per
        // lane).  Turning 32 x 32 tiles of the amplitudes through shared memory instead, so that lanes run along k_y, was
        // measured SLOWER on c5 (round 3: 211 vs 141 us per launch, 128 blocks): with one block per position the kernel is
        // latency-bound and the two barriers per tile cost more than the sector amplification, which L2 absorbs.
        for (int i = t; i < N * N; i += 256) {
            const int ky = i / N, kx = i - ky * N, ti = kx * N + ky;
            f(__ldg(Ib + ti), __ldg(ab + i), ti, i);
        }
    }
}

// a6 + a7, plain amplitude sum (north_star; reading R13), N = 64 / 256: L_b = sum_k (sqrt(I) - a)^2 and the seed
// weights w = 2 (1 - a / sqrt(I)) / N (0 where I = 0, R14) in the order of I; optionally I in natural order.  One block
// per position.
__global__ void __launch_bounds__(256) pty_loss_seed_kernel(const float* __restrict__ I, const float* __restrict__ a, int N,
                                                           double* loss, float* loss_per_pos, float* __restrict__ seed_w,
                                                           float* __restrict__ intensity) {
    __shared__ double part[8];
    const int b = blockIdx.x;
    const size_t NN = (size_t)N * N;
    float* Wb = seed_w + (size_t)b * NN;
    const float invN = 1.0f / (float)N;
    float acc = 0.f;
    float* out = intensity ? intensity + (size_t)b * NN : nullptr;
    sweep_position<false>(I + (size_t)b * NN, a + (size_t)b * NN, N, nullptr, [&](float iv, float av, int wi, int nat) {
        const float d = sqrtf(iv) - av;
        acc += d * d;
        Wb[wi] = iv > 1e-30f ? 2.0f * (1.0f - av * rsqrtf(iv)) * invN : 0.f;
        if (out) out[nat] = iv;
    });
    const double s = block_sum_256((double)acc, part);
    if (threadIdx.x == 0) {
        if (loss_per_pos) loss_per_pos[b] = (float)s;
        atomicAdd(loss, s);
    }
}

// Eq. 5-7, pass 1: the minibatch sums S = sum (sqrt(I) - a)^2, sum a, sum a^2, sum (a^2 log(I + eps) - I), and (PACBED)
// the position-summed patterns sum_b I_b(k), sum_b a_b(k)^2 in natural order.  One block per position.
template <bool TORD>
__global__ void __launch_bounds__(256) pty_loss_sums_kernel(const float* __restrict__ I, const float* __restrict__ a, int N,
                                                           LossCfg cfg, double* stats, float* loss_per_pos,
                                                           float* Isum, float* Imsum, float* __restrict__ intensity) {
    __shared__ float tile[TORD ? 32 : 1][129];
    __shared__ double part[8];
    const int b = blockIdx.x;
    const size_t NN = (size_t)N * N;
    float s = 0.f, sa = 0.f, sa2 = 0.f, sp = 0.f;
    const bool pacbed = cfg.w_pacbed != 0.f;
    float* out = intensity ? intensity + (size_t)b * NN : nullptr;
    sweep_position<TORD>(I + (size_t)b * NN, a + (size_t)b * NN, N, tile, [&](float iv, float av, int, int nat) {
        const float d = sqrtf(iv) - av, a2 = av * av;
        s += d * d; sa += av; sa2 += a2;
        sp += a2 * logf(iv + cfg.eps) - iv;
        if (pacbed) { red_add(Isum + nat, iv); red_add(Imsum + nat, a2); }
        if (out) out[nat] = iv;
    });
    const double S = block_sum_256((double)s, part), A = block_sum_256((double)sa, part),
                 A2 = block_sum_256((double)sa2, part), P = block_sum_256((double)sp, part);
    if (threadIdx.x == 0) {
        if (loss_per_pos) loss_per_pos[b] = (float)S;
        atomicAdd(stats + ST_S, S); atomicAdd(stats + ST_A, A); atomicAdd(stats + ST_A2, A2); atomicAdd(stats + ST_P, P);
    }
}

// Eq. 5-7 + Eq. 9, pass 2 (one block): the normalised terms, the total, and the coefficients of dL/dI:
//   dL/dI_b(k) = cG (1 - a / sqrt(I)) + cP (1 - a^2 / (I + eps)) + cPB (1 - sqrt(<I_meas>_B / <I>_B)).
// A minibatch whose measurements are all zero has no mean to normalise by (Eq. 5-7 divide by <a> and <a^2>): the terms
// and coefficients that would divide by zero are set to 0 and sticky flag bit 2 is raised (pty_status: PTY_ERR_ZERO_DATA).
__global__ void __launch_bounds__(256) pty_loss_finalize_kernel(int B, int N, LossCfg cfg, double* stats, const float* Isum,
                                                               const float* Imsum, double* loss, int* flags) {
    __shared__ double part[8];
    const double n = (double)B * N * N, nD = (double)N * N;
    double q = 0.0;
    if (cfg.w_pacbed != 0.f)
        for (int i = threadIdx.x; i < N * N; i += 256) {
            const double d = sqrt((double)Isum[i] / B) - sqrt((double)Imsum[i] / B);
            q += d * d;
        }
    const double Q = block_sum_256(q, part);
    if (threadIdx.x != 0) return;
    const double mean_a = stats[ST_A] / n, mse = stats[ST_S] / n, mean_im = stats[ST_A2] / n, mse_pb = Q / nD;
    const bool ok_a = mean_a != 0.0, ok_im = mean_im != 0.0;
    if (!ok_a || !ok_im) atomicOr(flags, 2);
    const double LG = ok_a ? sqrt(mse) / mean_a : 0.0, LP = ok_im ? -(stats[ST_P] / n) / mean_im : 0.0,
                 LPB = ok_a ? sqrt(mse_pb) / mean_a : 0.0;
    stats[ST_LG] = LG; stats[ST_LP] = LP; stats[ST_LPB] = LPB;
    stats[ST_CG] = (cfg.w_gaussian != 0.f && mse > 0.0 && ok_a) ? cfg.w_gaussian / (2.0 * sqrt(mse) * mean_a * n) : 0.0;
    stats[ST_CP] = (cfg.w_poisson != 0.f && ok_im) ? cfg.w_poisson / (n * mean_im) : 0.0;
    stats[ST_CPB] = (cfg.w_pacbed != 0.f && mse_pb > 0.0 && ok_a) ? cfg.w_pacbed / (2.0 * sqrt(mse_pb) * mean_a * nD * B) : 0.0;
    *loss = cfg.w_gaussian * LG + cfg.w_poisson * LP + cfg.w_pacbed * LPB + cfg.w_sparse * stats[ST_LS];
}

// pass 3: seed weights w = 2 (dL/dI) / N in the adjoint's order (the 1/N belongs to the unitary F^-1 of B2)
template <bool TORD>
__global__ void __launch_bounds__(256) pty_seed_kernel(const float* __restrict__ I, const float* __restrict__ a, int N, int B,
                                                      LossCfg cfg, const double* stats, const float* __restrict__ Isum,
                                                      const float* __restrict__ Imsum, float* __restrict__ seed_w) {
    __shared__ float tile[TORD ? 32 : 1][129];
    const int b = blockIdx.x;
    const size_t NN = (size_t)N * N;
    const float cG = (float)stats[ST_CG], cP = (float)stats[ST_CP], cPB = (float)stats[ST_CPB];
    const float k = 2.0f / (float)N;
    float* Wb = seed_w + (size_t)b * NN;
    sweep_position<TORD>(I + (size_t)b * NN, a + (size_t)b * NN, N, tile, [&](float iv, float av, int wi, int nat) {
        float d = cP * (1.0f - av * av / (iv + cfg.eps));
        if (iv > 1e-30f) d += cG * (1.0f - av * rsqrtf(iv));
        if (cPB != 0.f) {
            const float ib = __ldg(Isum + nat);
            if (ib > 1e-30f) d += cPB * (1.0f - sqrtf(__ldg(Imsum + nat) / ib));
        }
        Wb[wi] = k * d;
    });
}

// ------------------------------------------------------------------------------ amplitude / phase
__global__ void __launch_bounds__(256) pty_compose_object_kernel(const float* __restrict__ amp, const float* __restrict__ phase,
                                                                float2* __restrict__ obj, size_t n) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) {
        float s, c;
        sincosf(phase[i], &s, &c);
        const float A = amp[i];
        obj[i] = make_float2(A * c, A * s);
    }
}

// cnt[y][x] = number of patches of the minibatch that cover object pixel (y, x) (same crop origin as the big kernels)
__global__ void __launch_bounds__(256) pty_coverage_kernel(const float* __restrict__ positions, int N, int H, int W,
                                                          float* cnt) {
    const int b = blockIdx.x;
    const double py = (double)positions[2 * b], px = (double)positions[2 * b + 1];
    const int ry = min(max((int)floor(py + 0.5), 0), H - N), rx = min(max((int)floor(px + 0.5), 0), W - N);
    for (int i = threadIdx.x; i < N * N; i += 256) red_add(cnt + (size_t)(ry + i / N) * W + rx + i % N, 1.0f);
}

// Eq. 8, p = 1 (reading R27): sum over the patches of |phase| = sum over pixels of cnt |phase|
__global__ void __launch_bounds__(256) pty_sparse_sum_kernel(const float* __restrict__ phase, const float* __restrict__ cnt,
                                                            size_t n, size_t HW, double* stats) {
    __shared__ double part[8];
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256)
        acc += (double)(cnt[i % HW] * fabsf(phase[i]));
    const double s = block_sum_256(acc, part);
    if (threadIdx.x == 0) atomicAdd(stats + ST_SPARSE_SUM, s);
}
__global__ void pty_sparse_finalize_kernel(double* stats, double n_patch) { stats[ST_LS] = stats[ST_SPARSE_SUM] / n_patch; }

// chain rule of O = A exp(i phi) (R16): g_A = Re(conj(g_O) e^{i phi}), g_phi = Im(g_O conj(O)) + w4 dL_sparse/dphi
__global__ void __launch_bounds__(256) pty_amp_phase_grad_kernel(const float2* __restrict__ g_obj, const float* __restrict__ amp,
                                                                const float* __restrict__ phase, const float* __restrict__ cnt,
                                                                float c_sparse, size_t n, size_t HW, float* g_amp,
                                                                float* g_phase, int accumulate) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) {
        float s, c;
        const float ph = phase[i];
        sincosf(ph, &s, &c);
        const float2 g = g_obj[i];
        float ga = g.x * c + g.y * s;
        float gp = amp[i] * (g.y * c - g.x * s);
        if (c_sparse != 0.f) gp += c_sparse * cnt[i % HW] * (ph > 0.f ? 1.f : ph < 0.f ? -1.f : 0.f);
        if (accumulate) { ga += g_amp[i]; gp += g_phase[i]; }
        g_amp[i] = ga; g_phase[i] = gp;
    }
}

// ------------------------------------------------------------------------------ constraints (NEXT-3)
// Eq. 13: blur along depth, in place.  x is [outer][Nz][plane] floats; thread = one (outer, pixel) column, which walks
// z keeping the 2R + 1 ORIGINAL values it needs in registers; end slices replicated (reading R31).
// The taps travel BY VALUE as a kernel parameter: a launch (and a captured graph node) carries its own copy, so the call
// is enqueue-only with no host buffer that has to outlive it.
struct RzTaps { float t[17]; };
template <int R>
__global__ void __launch_bounds__(256) pty_rz_filter_kernel(float* x, int Nz, size_t plane, size_t columns, const RzTaps taps) {
    float g[2 * R + 1];
#pragma unroll
    for (int j = 0; j < 2 * R + 1; ++j) g[j] = taps.t[j];
    for (size_t col = (size_t)blockIdx.x * 256 + threadIdx.x; col < columns; col += (size_t)gridDim.x * 256) {
        float* p = x + (col / plane) * (size_t)Nz * plane + col % plane;
        float win[2 * R + 1];                        // win[j] = original x[clamp(z + j - R)]
        const float x0 = p[0];
#pragma unroll
        for (int j = 0; j < 2 * R + 1; ++j) win[j] = j <= R ? x0 : p[(size_t)min(j - R, Nz - 1) * plane];
        for (int z = 0; z < Nz; ++z) {
            float acc = 0.f;
#pragma unroll
            for (int j = 0; j < 2 * R + 1; ++j) acc += g[j] * win[j];
            p[(size_t)z * plane] = acc;
#pragma unroll
            for (int j = 0; j < 2 * R; ++j) win[j] = win[j + 1];
            const int zn = z + 1 + R;
            if (zn <= Nz - 1) win[2 * R] = p[(size_t)zn * plane];   // beyond the end: keep the (replicated) last slice
        }
    }
}

// positivity of the phase and amplitude clamp in one pass
__global__ void __launch_bounds__(256) pty_clip_clamp_kernel(float* amp, float* phase, size_t n, int phase_positive,
                                                            int clamp_amp, float lo, float hi) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) {
        if (phase_positive && phase) phase[i] = fmaxf(phase[i], 0.f);
        if (clamp_amp && amp) amp[i] = fminf(fmaxf(amp[i], lo), hi);
    }
}

// Probe-mode orthogonalisation (Thibault & Menzel 2013), three kernels.
// (1) Gram matrix G_ij = sum_r conj(P_i) P_j, one block per pair i <= j, double accumulation
__global__ void __launch_bounds__(256) pty_gram_kernel(const float2* __restrict__ probe, int M, size_t NN, double2* G) {
    __shared__ double part[8];
    int i = 0, j = 0, k = blockIdx.x;
    for (i = 0; i < M; ++i) { if (k < M - i) { j = i + k; break; } k -= M - i; }
    const float2* a = probe + (size_t)i * NN;
    const float2* b = probe + (size_t)j * NN;
    double re = 0.0, im = 0.0;
    for (size_t r = threadIdx.x; r < NN; r += 256) {
        const float2 x = a[r], y = b[r];
        re += (double)x.x * y.x + (double)x.y * y.y;
        im += (double)x.x * y.y - (double)x.y * y.x;
    }
    const double sr = block_sum_256(re, part), si = block_sum_256(im, part);
    if (threadIdx.x == 0) {
        G[i * M + j] = make_double2(sr, si);
        G[j * M + i] = make_double2(sr, -si);
    }
}

// (2) eigen-decomposition of the Hermitian M x M Gram matrix by cyclic complex Jacobi rotations (one thread; M <= 32):
// V's columns are the unit eigenvectors, ordered by decreasing eigenvalue; lam the eigenvalues.
constexpr int kMaxModes = 32;
__global__ void pty_eigh_kernel(const double2* G, int M, double2* V, double* lam) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    __shared__ double2 A[kMaxModes * kMaxModes], U[kMaxModes * kMaxModes];
    auto cmul_d = [](double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); };
    for (int k = 0; k < M * M; ++k) { A[k] = G[k]; U[k] = make_double2(k / M == k % M ? 1.0 : 0.0, 0.0); }
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = 0.0, tr = 0.0;
        for (int p = 0; p < M; ++p) {
            tr += fabs(A[p * M + p].x);
            for (int q = p + 1; q < M; ++q) off += A[p * M + q].x * A[p * M + q].x + A[p * M + q].y * A[p * M + q].y;
        }
        if (off <= 1e-30 * tr * tr) break;
        for (int p = 0; p < M; ++p)
            for (int q = p + 1; q < M; ++q) {
                const double2 apq = A[p * M + q];
                const double mag = sqrt(apq.x * apq.x + apq.y * apq.y);
                if (mag <= 1e-300) continue;
                const double2 ph = make_double2(apq.x / mag, apq.y / mag), phc = make_double2(ph.x, -ph.y);
                const double tau = (A[q * M + q].x - A[p * M + p].x) / (2.0 * mag);
                const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
                const double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
                for (int k = 0; k < M; ++k) {                     // columns p, q of A and of U
                    const double2 akp = A[k * M + p], akq = A[k * M + q];
                    const double2 x = cmul_d(phc, akq), y = cmul_d(ph, akp);
                    A[k * M + p] = make_double2(c * akp.x - s * x.x, c * akp.y - s * x.y);
                    A[k * M + q] = make_double2(s * y.x + c * akq.x, s * y.y + c * akq.y);
                    const double2 ukp = U[k * M + p], ukq = U[k * M + q];
                    const double2 xu = cmul_d(phc, ukq), yu = cmul_d(ph, ukp);
                    U[k * M + p] = make_double2(c * ukp.x - s * xu.x, c * ukp.y - s * xu.y);
                    U[k * M + q] = make_double2(s * yu.x + c * ukq.x, s * yu.y + c * ukq.y);
                }
                for (int k = 0; k < M; ++k) {                     // rows p, q of A
                    const double2 apk = A[p * M + k], aqk = A[q * M + k];
                    const double2 x = cmul_d(ph, aqk), y = cmul_d(phc, apk);
                    A[p * M + k] = make_double2(c * apk.x - s * x.x, c * apk.y - s * x.y);
                    A[q * M + k] = make_double2(s * y.x + c * aqk.x, s * y.y + c * aqk.y);
                }
            }
    }
    int order[kMaxModes];
    for (int k = 0; k < M; ++k) order[k] = k;
    for (int a = 0; a < M; ++a)                                    // selection sort, decreasing eigenvalue
        for (int b = a + 1; b < M; ++b)
            if (A[order[b] * M + order[b]].x > A[order[a] * M + order[a]].x) { const int t = order[a]; order[a] = order[b]; order[b] = t; }
    for (int k = 0; k < M; ++k) {
        lam[k] = fmax(A[order[k] * M + order[k]].x, 0.0);
        for (int j = 0; j < M; ++j) V[j * M + k] = U[j * M + order[k]];
    }
}

// (3) P'_k = sum_j V_jk P_j, in place: one thread per pixel holds all M values of that pixel
__global__ void __launch_bounds__(256) pty_mix_modes_kernel(float2* probe, int M, size_t NN, const double2* V) {
    __shared__ float2 Vs[kMaxModes * kMaxModes];
    for (int k = threadIdx.x; k < M * M; k += 256) Vs[k] = make_float2((float)V[k].x, (float)V[k].y);
    __syncthreads();
    for (size_t r = (size_t)blockIdx.x * 256 + threadIdx.x; r < NN; r += (size_t)gridDim.x * 256) {
        float2 in[kMaxModes];
        for (int j = 0; j < M; ++j) in[j] = probe[(size_t)j * NN + r];
        for (int k = 0; k < M; ++k) {
            float2 acc = make_float2(0.f, 0.f);
            for (int j = 0; j < M; ++j) {
                const float2 v = Vs[j * M + k];
                acc.x += v.x * in[j].x - v.y * in[j].y;
                acc.y += v.x * in[j].y + v.y * in[j].x;
            }
            probe[(size_t)k * NN + r] = acc;
        }
    }
}

}  // namespace pty
