// pty_lib.cu -- __global__ entry points, the small per-call kernels and the C ABI of include/pty.h.
// sm_100a only; no cuFFT, no CPU fallback: every step of the hot path runs in the kernels here.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/pty.h"
#include "pty_kernels.cuh"
#include "pty_kernels128.cuh"
#include "pty_kernels128g2.cuh"
#include "pty_pointwise.cuh"

namespace cg = cooperative_groups;
using namespace pty;

// ============================================================================ kernels
template <class SH>
__device__ __forceinline__ Cta<SH> make_cta(unsigned char* smem) {
    using I = ShapeInfo<SH>;
    Cta<SH> c;
    c.tid = threadIdx.x;
    c.rank = 0;
    c.S = reinterpret_cast<float2*>(smem);
    if constexpr (SH::CL > 1) {
        cg::cluster_group cl = cg::this_cluster();
        c.rank = (int)cl.block_rank();
#pragma unroll
        for (int k = 0; k < SH::CL; ++k) c.Sr[k] = cl.map_shared_rank(c.S, k);
    } else {
        c.Sr[0] = c.S;
    }
    float2* tab = reinterpret_cast<float2*>(smem + I::wave_bytes);
    c.tw = tab; c.Ey = tab + SH::N; c.Ex = tab + 2 * SH::N; c.My = tab + 3 * SH::N; c.Mx = tab + 4 * SH::N;
    c.red = reinterpret_cast<float*>(tab + 5 * SH::N);
    c.stg = reinterpret_cast<float2*>(smem + I::wave_bytes + I::table_bytes);
    c.rx = reinterpret_cast<unsigned long long*>(smem + I::wave_bytes + I::table_bytes + I::stage_bytes);
    c.rx_phase = 0;
    if constexpr (SH::CL > 1) {     // made visible to the peers by the cluster barrier that follows make_cta in the kernels
        if (threadIdx.x == 0) { mbar_init(c.rx, 1); mbar_init_fence(); }
    }
    return c;
}

template <class SH> struct MinBlocks { static constexpr int value = SH::N == 64 ? 2 : 1; };

template <class SH>
__global__ void __launch_bounds__(SH::NT, MinBlocks<SH>::value) pty_fwd_kernel(const KArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    Cta<SH> c = make_cta<SH>(smem);
    if constexpr (SH::CL > 1) cg::this_cluster().sync();
    fwd_body<SH>(A, c, blockIdx.x / SH::CL);
}

template <class SH>
__global__ void __launch_bounds__(SH::NT, MinBlocks<SH>::value) pty_bwd_kernel(const KArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    Cta<SH> c = make_cta<SH>(smem);
    if constexpr (SH::CL > 1) cg::this_cluster().sync();
    bwd_body<SH>(A, c, blockIdx.x / SH::CL);
}

// N = 128 helpers on the one-item register-resident FFT (pty_fft128.cuh): probe spectrum and probe gradient
__device__ __forceinline__ Cta128 make_cta128(unsigned char* smem) {
    Cta128 c;
    c.tid = threadIdx.x;
    c.X = reinterpret_cast<float2*>(smem);
    float2* tab = reinterpret_cast<float2*>(smem + F128::xch_bytes);
    c.twg = tab; c.Ey = tab + 128; c.Ex = tab + 256; c.My = tab + 384; c.Mx = tab + 512;
    c.red = reinterpret_cast<float*>(tab + 640);
    // tensor memory: all 512 columns, allocated by warp 0; thread (g, c) owns lane c, columns [128 g, +128)
    unsigned* tbase = reinterpret_cast<unsigned*>(c.red + 64);
    if ((threadIdx.x >> 5) == 0) tmem_alloc512(tbase);
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    c.tmq = *tbase + ((32u * ((threadIdx.x >> 5) & 3u)) << 16);
    return c;
}

__device__ __forceinline__ void release_cta128(unsigned char* smem) {
    tmem_fence_before_sync();
    __syncthreads();
    float2* tab = reinterpret_cast<float2*>(smem + F128::xch_bytes);
    if ((threadIdx.x >> 5) == 0) tmem_dealloc512(*reinterpret_cast<unsigned*>(reinterpret_cast<float*>(tab + 640) + 64));
}

// N = 128, two items per CTA (pty_kernels128g2.cuh): group G of CTA x owns item 2 x + G
// TMA: object rows staged by TMA (tmObj = the 3-D view of the object, make_object_map); false = register path only
// (odd W or an object pointer that is not 16-byte aligned, for which no tensor map exists).
template <bool HAT, bool TMA>
__global__ void __launch_bounds__(F128::NT, 1) pty_fwd128g2_kernel(const KArgs A, const __grid_constant__ CUtensorMap tmObj) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const G2 c = make_g2(smem);
    // persistent CTAs: TMEM allocation and the twiddle table once per SM; CTA x takes the item pairs x, x + grid, ...
    // (both groups run the same number of bodies: the hand-over of the transpose buffer is balanced per body)
    const int n = A.B * A.MT;
    G2Ring ring{};
    if constexpr (TMA) {
        ring = make_g2_ring(smem, c, &tmObj);
        if (ring.producer && 2 * (int)blockIdx.x < n) {      // the first role-step of this group's first item
            int row0, rx;
            g2_item_rows(A, min(2 * (int)blockIdx.x + c.G, n - 1), 2 * c.gg, row0, rx);
            g2_ring_fill(ring, rx, row0);
        }
    }
    for (int it = 2 * blockIdx.x; it < n; it += 2 * gridDim.x) {
        const int item = it + c.G;
        const int itn = it + 2 * (int)gridDim.x;
        fwd_body_g2<HAT, TMA>(A, c, ring, min(item, n - 1), item, item < n ? 1.f : 0.f,   // item == n: the ghost (slot n)
                              itn < n ? min(itn + c.G, n - 1) : -1);
        c.grp_sync();            // the next body rewrites the group's tables and reduction slots
    }
    release_g2(smem);
}
// PAIR: the two groups of a CTA sum their g_object contributions in shared memory before the one reduction (G2Pair;
// the host selects it only when every item pair 2x, 2x + 1 holds two modes of one position AND one object state,
// i.e. M is even: with an odd M and an even n_obj a pair would span two states, whose gradients are separate arrays)
template <bool HAT, bool PAIR> __global__ void __launch_bounds__(F128::NT, 1) pty_bwd128g2_kernel(const KArgs A) {
    extern __shared__ __align__(128) unsigned char smem[];
    const G2 c = make_g2(smem);
    G2Pair pr{};
    if constexpr (PAIR) pr = make_g2_pair(smem);
    const int n = A.B * A.MT;
    for (int it = 2 * blockIdx.x; it < n; it += 2 * gridDim.x) {
        int item = it + c.G;
        bwd_body_g2<HAT, PAIR>(A, c, pr, min(item, n - 1), item, item < n ? 1.f : 0.f);
        c.grp_sync();
    }
    release_g2(smem);
}

// a0: P^ = F[P] / N in thread order; a11: g_probe = F^-1[G^_P] / N (one CTA per mode)
__global__ void __launch_bounds__(F128::NT, 1) pty_probe_hat128_kernel(const float2* probe, float2* probe_hat_t) {
    extern __shared__ __align__(16) unsigned char smem[];
    probe_hat_body128(probe, probe_hat_t, make_cta128(smem), blockIdx.x);
    release_cta128(smem);
}
__global__ void __launch_bounds__(F128::NT, 1) pty_probe_grad128_kernel(const float2* GP_t, float2* g_probe, int accumulate) {
    extern __shared__ __align__(16) unsigned char smem[];
    probe_grad_body128(GP_t, g_probe, accumulate, make_cta128(smem), blockIdx.x);
    release_cta128(smem);
}

// a6 + a7 for N = 128: L_b = sum_k (sqrt(I_b) - a_b)^2 and the seed weights w = 2 (1 - a / sqrt(I)) / N
// (0 where I = 0, reading R14) written in the adjoint kernel's thread order
// [register r = 8 (kx >> 5) + (kx & 7)][tid = 128 ((kx >> 3) & 3) + ky].  I arrives in the forward kernel's thread
// order as pairs, [r / 2][128 o + ky][r & 1]; the measured amplitudes (natural order) are transposed through a
// 32-row shared tile so that both sides are coalesced; the natural-order copy of I (the optional `intensity`
// output of pty_forward_loss) is written from here.  One block of 256 threads per position.
__global__ void __launch_bounds__(256) pty_loss_seed128_kernel(const float* __restrict__ I, const float* __restrict__ a,
                                                              double* loss, float* loss_per_pos, float* __restrict__ seed_w,
                                                              float* __restrict__ intensity) {
    constexpr int N = 128;
    __shared__ float tile[32][N + 1];
    __shared__ double part[8];
    const int b = blockIdx.x, t = threadIdx.x;
    const float2* I2 = reinterpret_cast<const float2*>(I + (size_t)b * N * N);
    const float* ab = a + (size_t)b * N * N;
    float* Wb = seed_w + (size_t)b * N * N;
    float acc = 0.f;
    for (int ky0 = 0; ky0 < N; ky0 += 32) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int idx = j * 256 + t, row = idx >> 7, kx = idx & 127;
            tile[row][kx] = __ldg(ab + (ky0 + row) * N + kx);
        }
        __syncthreads();
        // one thread per (ky, pair of k_x): the pair (r, r + 1) of I is one 8-byte word, lanes along ky
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int idx = j * 256 + t, row = idx & 31, kx = 2 * (idx >> 5);
            const int r = 8 * (kx >> 5) + (kx & 7), g = (kx >> 3) & 3, ky = ky0 + row;
            const float2 iv = __ldg(I2 + (r >> 1) * 512 + 128 * g + ky);
            const float a0 = tile[row][kx], a1 = tile[row][kx + 1];
            const float d0 = sqrtf(iv.x) - a0, d1 = sqrtf(iv.y) - a1;
            acc += d0 * d0 + d1 * d1;
            Wb[r * 512 + 128 * g + ky] = iv.x > 1e-30f ? 2.0f * (1.0f - a0 * rsqrtf(iv.x)) * (1.0f / N) : 0.f;
            Wb[(r + 1) * 512 + 128 * g + ky] = iv.y > 1e-30f ? 2.0f * (1.0f - a1 * rsqrtf(iv.y)) * (1.0f / N) : 0.f;
            if (intensity) {
                float* o = intensity + (size_t)b * N * N + ky * N + kx;
                o[0] = iv.x; o[1] = iv.y;
            }
        }
        __syncthreads();
    }
    double dacc = (double)acc;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dacc += __shfl_xor_sync(0xffffffffu, dacc, o);
    if ((t & 31) == 0) part[t >> 5] = dacc;
    __syncthreads();
    if (t == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += part[w];
        if (loss_per_pos) loss_per_pos[b] = (float)s;
        atomicAdd(loss, s);
    }
}

template <class SH, int DIR>
__global__ void __launch_bounds__(SH::NT, MinBlocks<SH>::value)
pty_fft2_kernel(const float2* src, float2* dst, float scale, int accumulate) {
    extern __shared__ __align__(16) unsigned char smem[];
    Cta<SH> c = make_cta<SH>(smem);
    if constexpr (SH::CL > 1) cg::this_cluster().sync();
    fft2_body<SH, DIR>(src, dst, scale, accumulate, c, blockIdx.x / SH::CL);
}

// a0: separable propagator factors exp(i chi_y(k_y)), exp(i chi_x(k_x)) of Eq. 4 for one global tilt
// (PAPER.md:89): chi_a(k) = -pi lambda dz k^2 + 2 pi dz k tan(theta_a), k = fftfreq(N)/dx.  Double
// precision: 2N values per call.
__global__ void pty_prop_table_kernel(int N, float dz, float lambda, float dx, const float* tilt,
                                      float2* prop_y, float2* prop_x) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const double ty = tilt ? (double)tilt[0] : 0.0, tx = tilt ? (double)tilt[1] : 0.0;
    const double k = (double)(j < N / 2 ? j : j - N) / ((double)N * (double)dx);
    const double quad = -3.14159265358979323846 * (double)lambda * (double)dz * k * k;
    const double lin = 2.0 * 3.14159265358979323846 * (double)dz * k;
    const double chy = quad + lin * tan(ty), chx = quad + lin * tan(tx);
    prop_y[j] = make_float2((float)cos(chy), (float)sin(chy));
    prop_x[j] = make_float2((float)cos(chx), (float)sin(chx));
}

// a13 (B8): tilt and dz gradients from the per-position sums of D(k) (k in cycles/pixel).  One block; thread t
// handles positions t, t + 256, ...; the sums over b (global tilt, dz) are reduced in double precision.
__global__ void __launch_bounds__(256) pty_tilt_finalize_kernel(const float* dsum, const float* tilt, int B, int tilt_mode,
                                                                 float dz, float lambda, float dx, float* g_tilt, float* g_dz,
                                                                 int accumulate) {
    const double two_pi = 6.283185307179586476925;
    __shared__ double part[3][8];
    double gty = 0.0, gtx = 0.0, gz = 0.0;
    for (int b = threadIdx.x; b < B; b += blockDim.x) {
        double ty = 0.0, tx = 0.0;
        if (tilt_mode == 1) { ty = tilt[0]; tx = tilt[1]; }
        if (tilt_mode == 2) { ty = tilt[2 * b]; tx = tilt[2 * b + 1]; }
        const double sy = (double)dsum[4 * b] / dx, sx = (double)dsum[4 * b + 1] / dx;
        const double s2 = (double)dsum[4 * b + 2] / ((double)dx * dx);
        const double cy = cos(ty), cx = cos(tx);
        const double ay = two_pi * dz * sy / (cy * cy), ax = two_pi * dz * sx / (cx * cx);
        gz += -0.5 * two_pi * lambda * s2 + two_pi * (tan(tx) * sx + tan(ty) * sy);
        if (tilt_mode == 2 && g_tilt) {
            g_tilt[2 * b] = (accumulate ? g_tilt[2 * b] : 0.f) + (float)ay;
            g_tilt[2 * b + 1] = (accumulate ? g_tilt[2 * b + 1] : 0.f) + (float)ax;
        }
        gty += ay; gtx += ax;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        gty += __shfl_xor_sync(0xffffffffu, gty, o);
        gtx += __shfl_xor_sync(0xffffffffu, gtx, o);
        gz += __shfl_xor_sync(0xffffffffu, gz, o);
    }
    if ((threadIdx.x & 31) == 0) {
        part[0][threadIdx.x >> 5] = gty; part[1][threadIdx.x >> 5] = gtx; part[2][threadIdx.x >> 5] = gz;
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    gty = gtx = gz = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { gty += part[0][w]; gtx += part[1][w]; gz += part[2][w]; }
    if (tilt_mode == 1 && g_tilt) {
        g_tilt[0] = (accumulate ? g_tilt[0] : 0.f) + (float)gty;
        g_tilt[1] = (accumulate ? g_tilt[1] : 0.f) + (float)gtx;
    }
    if (g_dz) g_dz[0] = (accumulate ? g_dz[0] : 0.f) + (float)gz;
}

// a14 (B9): bias-corrected Adam on a flat float array.  HBM-bound: streams theta, g, m, v.
__global__ void __launch_bounds__(256) pty_adam_kernel(float* __restrict__ theta, const float* __restrict__ g,
                                                       float* __restrict__ m, float* __restrict__ v, size_t n,
                                                       size_t n4, float lr, float b1, float b2, float omb1, float omb2,
                                                       float eps, float inv_bc1, float inv_bc2) {
    // n4 = number of leading float4 groups (n / 4, or 0 when some array is not 16-byte aligned: scalar path)
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    float4* t4 = reinterpret_cast<float4*>(theta);
    const float4* g4 = reinterpret_cast<const float4*>(g);
    float4* m4 = reinterpret_cast<float4*>(m);
    float4* v4 = reinterpret_cast<float4*>(v);
    auto upd = [&](float& th, float gg, float& mm, float& vv) {
        mm = b1 * mm + omb1 * gg;
        vv = b2 * vv + omb2 * gg * gg;
        th -= lr * (mm * inv_bc1) / (sqrtf(vv * inv_bc2) + eps);
    };
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
        float4 th = t4[i], gg = __ldg(g4 + i), mm = m4[i], vv = v4[i];
        upd(th.x, gg.x, mm.x, vv.x); upd(th.y, gg.y, mm.y, vv.y);
        upd(th.z, gg.z, mm.z, vv.z); upd(th.w, gg.w, mm.w, vv.w);
        t4[i] = th; m4[i] = mm; v4[i] = vv;
    }
    for (size_t i = n4 * 4 + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        float th = theta[i], mm = m[i], vv = v[i];
        upd(th, g[i], mm, vv);
        theta[i] = th; m[i] = mm; v[i] = vv;
    }
}

// ============================================================================ host side
namespace {

thread_local std::string g_create_error;

struct Layout {
    size_t probe_hat, prop, I, ws_psi, ws_Psi, ws_hat, GP_hat, dsum, seed_w, scalars;
    size_t stats, Isum, Imsum, taps, gram, eigv, eigl;       // loss family (Eq. 5-9) and constraints
    size_t ap_object, ap_g_object, ap_cnt;                    // PTY_FLAG_AMP_PHASE
    size_t g_object, g_probe, g_pos, g_tilt;               // PTY_FLAG_STEP / PTY_FLAG_HOST
    size_t h_object, h_probe, h_pos, h_tilt, h_meas;       // PTY_FLAG_HOST staging
    size_t total;
};

size_t align_up(size_t x) { return (x + 255) & ~size_t(255); }

bool save_hat_of(const pty_dims& d) { return d.Nz > 1 && (d.tilt_mode != 0 || (d.flags & PTY_FLAG_SPECTRA)); }

int n_obj_of(const pty_dims& d) { return d.n_obj > 1 ? d.n_obj : 1; }

int validate_dims(const pty_dims* d, std::string& err) {
    if (!d) { err = "dims is null"; return PTY_ERR_INVALID_ARG; }
    if (d->n_obj < 0 || d->n_obj > 64) { err = "n_obj must be in [0, 64]"; return PTY_ERR_INVALID_ARG; }
    if (d->Nz < 1 || d->M < 1 || d->Bmax < 1 || d->H < 1 || d->W < 1) { err = "non-positive dimension"; return PTY_ERR_INVALID_ARG; }
    if (d->tilt_mode < 0 || d->tilt_mode > 2) { err = "tilt_mode must be 0, 1 or 2"; return PTY_ERR_INVALID_ARG; }
    if (!(d->dx > 0.f) || !(d->lambda >= 0.f)) { err = "dx must be > 0 and lambda >= 0"; return PTY_ERR_INVALID_ARG; }
    if (d->N != 64 && d->N != 128 && d->N != 256) { err = "N must be 64, 128 or 256"; return PTY_ERR_UNSUPPORTED; }
    if (d->N > d->H || d->N > d->W) { err = "probe window larger than the object"; return PTY_ERR_UNSUPPORTED; }
    return PTY_OK;
}

Layout make_layout(const pty_dims& d) {
    Layout L{};
    const size_t NN = (size_t)d.N * d.N, B = (size_t)d.Bmax, M = (size_t)d.M, Nz = (size_t)d.Nz;
    const size_t MT = M * (size_t)n_obj_of(d);       // waves per position: probe modes x object states
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
    L.probe_hat = take(M * NN * 8);
    L.prop = take(2 * (size_t)d.N * 8);
    L.I = take(B * NN * 4);
    // + 1: the spare slot of the N = 128 kernels' ghost item (odd item counts)
    L.ws_psi = take((B * MT + 1) * Nz * NN * 8);
    L.ws_Psi = take((B * MT + 1) * NN * 8);
    L.ws_hat = take(save_hat_of(d) ? (B * MT + 1) * (Nz - 1) * NN * 8 : 0);
    L.GP_hat = take(M * NN * 8);
    L.dsum = take(B * 4 * 4);
    L.seed_w = take(B * NN * 4);
    L.scalars = take(256);
    L.stats = take(ST_COUNT * sizeof(double));
    L.Isum = take(NN * 4);
    L.Imsum = take(NN * 4);
    L.taps = take(17 * 4);
    L.gram = take(M * M * 16);
    L.eigv = take(M * M * 16);
    L.eigl = take(M * 8);
    const bool grads = d.flags & (PTY_FLAG_STEP | PTY_FLAG_HOST);
    const size_t obj = (size_t)n_obj_of(d) * Nz * (size_t)d.H * d.W * 8;
    const bool ap = d.flags & PTY_FLAG_AMP_PHASE;
    L.ap_object = take(ap ? obj : 0);
    L.ap_g_object = take(ap ? obj : 0);
    L.ap_cnt = take(ap ? (size_t)d.H * d.W * 4 : 0);
    L.g_object = take(grads ? obj : 0);
    L.g_probe = take(grads ? M * NN * 8 : 0);
    L.g_pos = take(grads ? B * 2 * 4 : 0);
    L.g_tilt = take(grads ? B * 2 * 4 + 16 : 0);
    const bool host = d.flags & PTY_FLAG_HOST;
    L.h_object = take(host ? obj : 0);
    L.h_probe = take(host ? M * NN * 8 : 0);
    L.h_pos = take(host ? B * 2 * 4 : 0);
    L.h_tilt = take(host ? B * 2 * 4 + 16 : 0);
    L.h_meas = take(host ? B * NN * 4 : 0);
    L.total = off;
    return L;
}

}  // namespace

struct pty_plan {
    pty_dims d;
    Layout L;
    unsigned char* ws;
    int device;
    int num_sms;
    std::string err;
    cudaStream_t last_stream;
    int64_t launches;
    // state left by the last forward
    bool fwd_valid;
    const void *f_object, *f_probe, *f_positions, *f_tilt, *f_meas;
    int32_t f_B;

    CUtensorMap tm_obj;          // TMA view of the object last seen by a forward / adjoint launch (object_map)
    const void* tm_obj_ptr;
    pty_loss loss_cfg;           // pty_set_loss; mode 0 = plain amplitude sum
    bool sparse_ready;           // the AP forward has put L_sparse into the statistics of this call
    // pty_grad_host: the measurements travel on a second stream while the forward kernel runs (only the loss reads them)
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_in = nullptr, ev_meas = nullptr;
    bool wait_meas = false;
    // optional kernel timing (pty_profile)
    bool profiling;
    struct Timed { cudaEvent_t a, b; int which; };
    std::vector<Timed> timed;

    template <class T> T* at(size_t off) const { return reinterpret_cast<T*>(ws + off); }
    double* d_loss() const { return at<double>(L.scalars); }
    int* d_flags() const { return at<int>(L.scalars + 64); }
    float* d_gdz() const { return at<float>(L.scalars + 128); }
    double* d_stats() const { return at<double>(L.stats); }
    int n_obj() const { return d.n_obj > 1 ? d.n_obj : 1; }
    size_t object_elems() const { return (size_t)n_obj() * d.Nz * d.H * d.W; }
    LossCfg loss_dev() const { return LossCfg{loss_cfg.w_gaussian, loss_cfg.w_poisson, loss_cfg.w_pacbed, loss_cfg.w_sparse, loss_cfg.eps}; }
};

namespace {

int fail(pty_plan* p, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (p) p->err = buf; else g_create_error = buf;
    return code;
}

// Every entry point runs on the plan's device whatever the caller's current device is, and restores it.
struct DeviceGuard {
    int prev; bool switched;
    explicit DeviceGuard(int device) : prev(-1), switched(false) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

#define PTY_CUDA(p, call)                                                                     \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(p, PTY_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                        __FILE__, __LINE__);                                                  \
    } while (0)

template <class K, class... Args>
cudaError_t launch(pty_plan* p, K kernel, int grid, int block, size_t smem, int cluster, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    int na = 0;
    if (cluster > 1) {
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = (unsigned)cluster;
        attr[na].val.clusterDim.y = 1;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    p->launches++;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}

template <class SH> cudaError_t set_smem_attrs() {
    const int bytes = (int)ShapeInfo<SH>::smem_bytes;
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(pty_fwd_kernel<SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))) return e;
    if ((e = cudaFuncSetAttribute(pty_bwd_kernel<SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))) return e;
    if ((e = cudaFuncSetAttribute(pty_fft2_kernel<SH, -1>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))) return e;
    if ((e = cudaFuncSetAttribute(pty_fft2_kernel<SH, +1>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes))) return e;
    return cudaSuccess;
}

template <class SH> cudaError_t launch_fft2(pty_plan* p, int dir, const float2* src, float2* dst, float scale, int acc, int items, cudaStream_t st) {
    const size_t smem = ShapeInfo<SH>::smem_bytes;
    if (dir < 0) return launch(p, pty_fft2_kernel<SH, -1>, items * SH::CL, SH::NT, smem, SH::CL, st, src, dst, scale, acc);
    return launch(p, pty_fft2_kernel<SH, +1>, items * SH::CL, SH::NT, smem, SH::CL, st, src, dst, scale, acc);
}
// brackets one launch with events when pty_profile is on
struct ScopedTimer {
    pty_plan* p; cudaStream_t st; pty_plan::Timed t; bool on;
    ScopedTimer(pty_plan* p_, int which, cudaStream_t st_) : p(p_), st(st_), on(false) {
        if (!p->profiling || p->timed.size() >= 1024) return;
        if (cudaEventCreate(&t.a) != cudaSuccess) return;
        if (cudaEventCreate(&t.b) != cudaSuccess) { cudaEventDestroy(t.a); return; }
        t.which = which; on = true;
        cudaEventRecord(t.a, st);
    }
    ~ScopedTimer() {
        if (!on) return;
        cudaEventRecord(t.b, st);
        p->timed.push_back(t);
    }
};

// N = 128 runs the two-items-per-CTA kernels (pty_kernels128g2.cuh); N = 64 and N = 256 the shared-memory passes
template <class SH> cudaError_t launch_fwd_sh(pty_plan* p, const KArgs& A, cudaStream_t st) {
    return launch(p, pty_fwd_kernel<SH>, A.B * A.MT * SH::CL, SH::NT, ShapeInfo<SH>::smem_bytes, SH::CL, st, A);
}
template <class SH> cudaError_t launch_bwd_sh(pty_plan* p, const KArgs& A, cudaStream_t st) {
    return launch(p, pty_bwd_kernel<SH>, A.B * A.MT * SH::CL, SH::NT, ShapeInfo<SH>::smem_bytes, SH::CL, st, A);
}
// ---- the object as a TMA tensor (G2Ring): 3-D view (x, row % 4, row / 4) of 8-byte elements, box {130, 1, 4}.
// cuTensorMapEncodeTiled comes from the driver through the runtime (no link against libcuda).  The map is cached per
// object pointer; TMA needs a 16-byte aligned base and row pitch, otherwise the register path runs.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            f = nullptr;
        return reinterpret_cast<EncodeTiledFn>(f);
    }();
    return fn;
}
// true when `object` can be read through TMA; fills p->tm_obj (cached)
bool object_map(pty_plan* p, const void* object) {
    const pty_dims& d = p->d;
    if (d.N != 128 || (d.W & 1) || (reinterpret_cast<uintptr_t>(object) & 15) || !(p->d.flags & PTY_FLAG_TMA_OBJECT)) return false;
    if (p->tm_obj_ptr == object) return true;
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const cuuint64_t rows = (cuuint64_t)p->n_obj() * d.Nz * d.H;
    const cuuint64_t dims[3] = {(cuuint64_t)d.W, 4, (rows + 3) / 4};
    const cuuint64_t strides[2] = {(cuuint64_t)d.W * 8, (cuuint64_t)d.W * 32};     // bytes, dims 1 and 2
    const cuuint32_t box[3] = {(cuuint32_t)G2Ring::COLS, 1, (cuuint32_t)G2Ring::ROWS};
    const cuuint32_t estr[3] = {1, 1, 1};
    if (enc(&p->tm_obj, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(object), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    p->tm_obj_ptr = object;
    return true;
}

int g2_grid(const pty_plan* p, const KArgs& A) {      // one persistent CTA per SM, or fewer when there is less work
    const int pairs = (A.B * A.MT + 1) / 2;
    return pairs < p->num_sms ? pairs : p->num_sms;
}
cudaError_t launch_fwd(pty_plan* p, const KArgs& A, cudaStream_t st) {
    ScopedTimer tm(p, 0, st);
    if (p->d.N == 128) {
        const int grid = g2_grid(p, A);
        if (object_map(p, A.object))
            return A.save_hat ? launch(p, pty_fwd128g2_kernel<true, true>, grid, F128::NT, G2Ring::bytes, 1, st, A, p->tm_obj)
                              : launch(p, pty_fwd128g2_kernel<false, true>, grid, F128::NT, G2Ring::bytes, 1, st, A, p->tm_obj);
        return A.save_hat ? launch(p, pty_fwd128g2_kernel<true, false>, grid, F128::NT, G2Smem::bytes, 1, st, A, p->tm_obj)
                          : launch(p, pty_fwd128g2_kernel<false, false>, grid, F128::NT, G2Smem::bytes, 1, st, A, p->tm_obj);
    }
    return p->d.N == 64 ? launch_fwd_sh<Shape<64>>(p, A, st) : launch_fwd_sh<Shape<256>>(p, A, st);
}
cudaError_t launch_bwd(pty_plan* p, const KArgs& A, cudaStream_t st) {
    ScopedTimer tm(p, 1, st);
    if (p->d.N == 128)
    {
        if ((p->d.flags & PTY_FLAG_PAIR_SUM) && A.M % 2 == 0)    // item = (b n_obj + n) M + m: an even M keeps a pair in one (b, n)
            return A.save_hat ? launch(p, pty_bwd128g2_kernel<true, true>, g2_grid(p, A), F128::NT, G2Pair::bytes, 1, st, A)
                              : launch(p, pty_bwd128g2_kernel<false, true>, g2_grid(p, A), F128::NT, G2Pair::bytes, 1, st, A);
        return A.save_hat ? launch(p, pty_bwd128g2_kernel<true, false>, g2_grid(p, A), F128::NT, G2Smem::bytes, 1, st, A)
                          : launch(p, pty_bwd128g2_kernel<false, false>, g2_grid(p, A), F128::NT, G2Smem::bytes, 1, st, A);
    }
    return p->d.N == 64 ? launch_bwd_sh<Shape<64>>(p, A, st) : launch_bwd_sh<Shape<256>>(p, A, st);
}
// plain 2-D FFT of `items` planes (N = 64, 256): P^ = F[P] / N and g_probe = F^-1[G^_P] / N
cudaError_t launch_fft2_n(pty_plan* p, int dir, const float2* src, float2* dst, float scale, int acc, int items, cudaStream_t st) {
    return p->d.N == 64 ? launch_fft2<Shape<64>>(p, dir, src, dst, scale, acc, items, st)
                        : launch_fft2<Shape<256>>(p, dir, src, dst, scale, acc, items, st);
}

KArgs make_args(const pty_plan* p, const void* object, const float* positions, const float* tilt,
                const float* meas, int32_t B) {
    KArgs A{};
    const pty_dims& d = p->d;
    A.Nz = d.Nz; A.H = d.H; A.W = d.W; A.M = d.M; A.B = B;
    A.Nobj = p->n_obj(); A.MT = d.M * A.Nobj;
    A.tilt_mode = d.tilt_mode;
    A.save_hat = save_hat_of(d) ? 1 : 0;
    A.dz = d.dz; A.lambda = d.lambda; A.dx = d.dx;
    A.object = static_cast<const float2*>(object);
    A.probe_hat = p->at<float2>(p->L.probe_hat);
    A.positions = positions;
    A.tilt = tilt;
    A.meas = meas;
    A.prop_y = p->at<float2>(p->L.prop);
    A.prop_x = p->at<float2>(p->L.prop) + d.N;
    A.I = p->at<float>(p->L.I);
    A.ws_psi = p->at<float2>(p->L.ws_psi);
    A.ws_Psi = p->at<float2>(p->L.ws_Psi);
    A.ws_hat = A.save_hat ? p->at<float2>(p->L.ws_hat) : nullptr;
    A.GP_hat = p->at<float2>(p->L.GP_hat);
    A.dsum = p->at<float>(p->L.dsum);
    A.seed_w = p->at<float>(p->L.seed_w);
    A.flags = p->d_flags();
    return A;
}

int check_batch(pty_plan* p, const void* object, const void* probe, const float* positions, const float* tilt,
                const float* meas, int32_t B) {
    if (!p) return PTY_ERR_INVALID_ARG;
    if (!object || !probe || (B > 0 && (!positions || !meas))) return fail(p, PTY_ERR_INVALID_ARG, "null input pointer");
    if (p->d.tilt_mode != 0 && !tilt) return fail(p, PTY_ERR_INVALID_ARG, "tilt_mode %d needs a tilt pointer", p->d.tilt_mode);
    if (B < 0 || B > p->d.Bmax) return fail(p, PTY_ERR_INVALID_ARG, "B = %d outside [0, Bmax = %d]", B, p->d.Bmax);
    // complex arrays are read as 8-byte words, the measured amplitudes as 16-byte vectors (pty.h "Alignment")
    if ((reinterpret_cast<uintptr_t>(object) & 7) || (reinterpret_cast<uintptr_t>(probe) & 7))
        return fail(p, PTY_ERR_INVALID_ARG, "object and probe must be 8-byte aligned");
    if (reinterpret_cast<uintptr_t>(meas) & 15)
        return fail(p, PTY_ERR_INVALID_ARG, "meas_amp must be 16-byte aligned");
    if ((reinterpret_cast<uintptr_t>(positions) & 3) || (reinterpret_cast<uintptr_t>(tilt) & 3))
        return fail(p, PTY_ERR_INVALID_ARG, "positions and tilt must be 4-byte aligned");
    return PTY_OK;
}

// a0 + a2..a6 for one minibatch
int run_forward(pty_plan* p, const void* object, const void* probe, const float* positions, const float* tilt,
                const float* meas, int32_t B, double* loss, float* loss_per_pos, float* intensity, cudaStream_t st) {
    const pty_dims& d = p->d;
    const size_t NN = (size_t)d.N * d.N;
    p->last_stream = st;
    p->fwd_valid = false;
    // one-shot hand-overs from ap_prepare / pty_grad_host: taken and cleared here so that no exit path (B == 0, a CUDA
    // error) leaves them set for the next, unrelated call on this plan
    const bool sparse_ready = p->sparse_ready, wait_meas = p->wait_meas;
    p->sparse_ready = false;
    p->wait_meas = false;
    PTY_CUDA(p, cudaMemsetAsync(loss, 0, sizeof(double), st));
    if (B == 0) {
        if (wait_meas) PTY_CUDA(p, cudaStreamWaitEvent(st, p->ev_meas, 0));
        return PTY_OK;
    }
    const bool paper_loss = p->loss_cfg.mode == 1;
    if (paper_loss) {   // the minibatch sums of Eq. 5-7 (the AP entry point has already put L_sparse in place)
        if (!sparse_ready) PTY_CUDA(p, cudaMemsetAsync(p->d_stats(), 0, ST_COUNT * sizeof(double), st));
        else PTY_CUDA(p, cudaMemsetAsync(p->d_stats(), 0, 4 * sizeof(double), st));
        if (p->loss_cfg.w_pacbed != 0.f) {
            PTY_CUDA(p, cudaMemsetAsync(p->at<float>(p->L.Isum), 0, NN * sizeof(float), st));
            PTY_CUDA(p, cudaMemsetAsync(p->at<float>(p->L.Imsum), 0, NN * sizeof(float), st));
        }
    }
    KArgs A = make_args(p, object, positions, tilt, meas, B);
    // a0: probe spectrum (unitary) and propagator factors
    if (d.N == 128)
        PTY_CUDA(p, launch(p, pty_probe_hat128_kernel, d.M, F128::NT, F128::smem_bytes, 1, st, (const float2*)probe, p->at<float2>(p->L.probe_hat)));
    else
        PTY_CUDA(p, launch_fft2_n(p, -1, (const float2*)probe, p->at<float2>(p->L.probe_hat), 1.f / d.N, 0, d.M, st));
    if (d.tilt_mode != 2)
        PTY_CUDA(p, launch(p, pty_prop_table_kernel, (d.N + 127) / 128, 128, 0, 1, st, (int)d.N, d.dz, d.lambda, d.dx,
                           d.tilt_mode == 1 ? tilt : (const float*)nullptr, p->at<float2>(p->L.prop), p->at<float2>(p->L.prop) + d.N));
    PTY_CUDA(p, cudaMemsetAsync(A.I, 0, (size_t)B * NN * sizeof(float), st));
    PTY_CUDA(p, launch_fwd(p, A, st));
    if (wait_meas)           // pty_grad_host: the loss is the first reader of the measurements
        PTY_CUDA(p, cudaStreamWaitEvent(st, p->ev_meas, 0));
    if (paper_loss) {
        const LossCfg cfg = p->loss_dev();
        float* Isum = p->at<float>(p->L.Isum);
        float* Imsum = p->at<float>(p->L.Imsum);
        if (d.N == 128) {
            PTY_CUDA(p, launch(p, pty_loss_sums_kernel<true>, B, 256, 0, 1, st, (const float*)A.I, meas, (int)d.N, cfg, p->d_stats(), loss_per_pos, Isum, Imsum, intensity));
            PTY_CUDA(p, launch(p, pty_loss_finalize_kernel, 1, 256, 0, 1, st, (int)B, (int)d.N, cfg, p->d_stats(), (const float*)Isum, (const float*)Imsum, loss, p->d_flags()));
            PTY_CUDA(p, launch(p, pty_seed_kernel<true>, B, 256, 0, 1, st, (const float*)A.I, meas, (int)d.N, (int)B, cfg, (const double*)p->d_stats(), (const float*)Isum, (const float*)Imsum, A.seed_w));
        } else {
            PTY_CUDA(p, launch(p, pty_loss_sums_kernel<false>, B, 256, 0, 1, st, (const float*)A.I, meas, (int)d.N, cfg, p->d_stats(), loss_per_pos, Isum, Imsum, intensity));
            PTY_CUDA(p, launch(p, pty_loss_finalize_kernel, 1, 256, 0, 1, st, (int)B, (int)d.N, cfg, p->d_stats(), (const float*)Isum, (const float*)Imsum, loss, p->d_flags()));
            PTY_CUDA(p, launch(p, pty_seed_kernel<false>, B, 256, 0, 1, st, (const float*)A.I, meas, (int)d.N, (int)B, cfg, (const double*)p->d_stats(), (const float*)Isum, (const float*)Imsum, A.seed_w));
        }
    } else if (d.N == 128) {
        PTY_CUDA(p, launch(p, pty_loss_seed128_kernel, B, 256, 0, 1, st, (const float*)A.I, meas, loss, loss_per_pos, A.seed_w, intensity));
    } else {
        PTY_CUDA(p, launch(p, pty_loss_seed_kernel, B, 256, 0, 1, st, (const float*)A.I, meas, (int)d.N, loss, loss_per_pos, A.seed_w, intensity));
    }
    p->fwd_valid = true;
    p->f_object = object; p->f_probe = probe; p->f_positions = positions; p->f_tilt = tilt; p->f_meas = meas;
    p->f_B = B;
    return PTY_OK;
}

// a7..a13 for one minibatch; needs the forward state
int run_backward(pty_plan* p, const void* object, const float* positions, const float* tilt, const float* meas,
                 int32_t B, void* g_object, void* g_probe, float* g_positions, float* g_tilt, float* g_dz,
                 int accumulate, cudaStream_t st, int accumulate_object = -1) {
    // accumulate: add into g_probe, g_positions, g_tilt, g_dz; accumulate_object (default: the same) into g_object
    const pty_dims& d = p->d;
    const size_t NN = (size_t)d.N * d.N;
    p->last_stream = st;
    if (accumulate_object < 0) accumulate_object = accumulate;
    if (!accumulate_object) PTY_CUDA(p, cudaMemsetAsync(g_object, 0, p->object_elems() * sizeof(float2), st));
    if (!accumulate && g_positions && B) PTY_CUDA(p, cudaMemsetAsync(g_positions, 0, (size_t)B * 2 * sizeof(float), st));
    KArgs A = make_args(p, object, positions, tilt, meas, B);
    A.g_object = static_cast<float2*>(g_object);
    A.g_pos = g_positions;
    const bool want_probe = g_probe != nullptr;
    PTY_CUDA(p, cudaMemsetAsync(A.GP_hat, 0, (size_t)d.M * NN * sizeof(float2), st));
    if (A.save_hat && B) PTY_CUDA(p, cudaMemsetAsync(A.dsum, 0, (size_t)B * 4 * sizeof(float), st));
    if (B)
        PTY_CUDA(p, launch_bwd(p, A, st));
    if (want_probe && d.N == 128)
        PTY_CUDA(p, launch(p, pty_probe_grad128_kernel, d.M, F128::NT, F128::smem_bytes, 1, st, (const float2*)A.GP_hat, (float2*)g_probe, (int)accumulate));
    else if (want_probe)
        PTY_CUDA(p, launch_fft2_n(p, +1, A.GP_hat, (float2*)g_probe, 1.f / d.N, accumulate, d.M, st));
    const bool want_tilt = g_tilt && d.tilt_mode != 0;
    if (want_tilt || g_dz) {
        if (A.save_hat) {
            PTY_CUDA(p, launch(p, pty_tilt_finalize_kernel, 1, 256, 0, 1, st, (const float*)A.dsum, tilt, (int)B, (int)d.tilt_mode,
                               d.dz, d.lambda, d.dx, want_tilt ? g_tilt : (float*)nullptr, g_dz, accumulate));
        } else if (!accumulate) {   // Nz == 1: no propagation, so both gradients are exactly zero
            if (want_tilt) PTY_CUDA(p, cudaMemsetAsync(g_tilt, 0, (d.tilt_mode == 2 ? (size_t)B * 2 : 2) * sizeof(float), st));
            if (g_dz) PTY_CUDA(p, cudaMemsetAsync(g_dz, 0, sizeof(float), st));
        }
    }
    return PTY_OK;
}

int adam_launch(pty_plan* p, float* theta, const float* g, float* m, float* v, size_t n, float lr, float b1, float b2,
                float eps, int32_t t, cudaStream_t st) {
    if (n == 0 || lr == 0.f) return PTY_OK;
    if (!theta || !g || !m || !v) return fail(p, PTY_ERR_INVALID_ARG, "adam: null pointer");
    if (t < 1) return fail(p, PTY_ERR_INVALID_ARG, "adam: step number t must be >= 1");
    const float inv_bc1 = (float)(1.0 / (1.0 - pow((double)b1, (double)t)));
    const float inv_bc2 = (float)(1.0 / (1.0 - pow((double)b2, (double)t)));
    const bool aligned = ((reinterpret_cast<uintptr_t>(theta) | reinterpret_cast<uintptr_t>(g) |
                           reinterpret_cast<uintptr_t>(m) | reinterpret_cast<uintptr_t>(v)) & 15) == 0;
    const size_t n4 = aligned ? n / 4 : 0;      // e.g. a positions[lo:hi] view with odd lo: scalar path
    size_t blocks = ((aligned ? n / 4 : n) + 255) / 256;
    const size_t cap = (size_t)p->num_sms * 16;
    if (blocks > cap) blocks = cap;
    if (blocks == 0) blocks = 1;
    const float omb1 = (float)(1.0 - (double)b1), omb2 = (float)(1.0 - (double)b2);   // 1 - beta rounded once
    PTY_CUDA(p, launch(p, pty_adam_kernel, (int)blocks, 256, 0, 1, st, theta, g, m, v, n, n4, lr, b1, b2, omb1, omb2, eps,
                       inv_bc1, inv_bc2));
    return PTY_OK;
}

}  // namespace

// ---------------------------------------------------------------------------- scratch of pty_ortho_probe_noalloc
// The one piece of device memory this library owns: Gram matrix, eigenvectors and eigenvalues of the probe-mode
// orthogonalisation for callers that cannot hand over a workspace (include/pty.h).  It is part of the module's
// device image, so every GPU that loads the module holds these 33,024 bytes until the process exits.
// In HOST code the name below is only a handle for the runtime's symbol calls, not a device address: handing it to a
// kernel would make the kernel fault, or, where the GPU can reach host memory, read and write the wrong memory without
// a fault.  noalloc_scratch() asks the runtime for the real address on each device and only that goes to the kernels.
static_assert(PTY_ORTHO_NOALLOC_MAX_MODES == pty::kMaxModes, "pty.h and the eigen-solver disagree on the mode limit");
static __device__ __align__(256) unsigned char g_ortho_noalloc_scratch[PTY_ORTHO_NOALLOC_SCRATCH_BYTES];

namespace {
constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mutex;
unsigned char* g_noalloc_addr[kNoAllocMaxDevices];      // device address of the array on device i; null = not asked yet

// Address of the scratch array on `device`, which the caller has made current.  The first call per device asks the
// runtime (this is the set-up step pty.h tells callers to run before any stream capture); later calls read the table.
int noalloc_scratch(int device, unsigned char** out) {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_addr[device]) {
        unsigned char* ptr = nullptr;
        PTY_CUDA(nullptr, cudaGetSymbolAddress((void**)&ptr, g_ortho_noalloc_scratch));
        if (!ptr) return fail(nullptr, PTY_ERR_CUDA, "cudaGetSymbolAddress returned a null scratch address on device %d", device);
        g_noalloc_addr[device] = ptr;
    }
    *out = g_noalloc_addr[device];
    return PTY_OK;
}
}  // namespace

// ============================================================================ C ABI
extern "C" {

const char* pty_version(void) { return "pty-b200 0.2 (sm_100a)"; }

int pty_workspace_bytes(const pty_dims* dims, size_t* out_bytes) {
    std::string err;
    int rc = validate_dims(dims, err);
    if (rc != PTY_OK) { g_create_error = err; return rc; }
    if (!out_bytes) { g_create_error = "out_bytes is null"; return PTY_ERR_INVALID_ARG; }
    *out_bytes = make_layout(*dims).total;
    return PTY_OK;
}

int pty_create(pty_plan** out_plan, const pty_dims* dims, void* workspace, size_t workspace_bytes, int device) {
    if (!out_plan) { g_create_error = "out_plan is null"; return PTY_ERR_INVALID_ARG; }
    *out_plan = nullptr;
    std::string err;
    int rc = validate_dims(dims, err);
    if (rc != PTY_OK) { g_create_error = err; return rc; }
    Layout L = make_layout(*dims);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255) != 0 || workspace_bytes < L.total)
        return fail(nullptr, PTY_ERR_WORKSPACE, "workspace null, not 256-byte aligned or smaller than %zu bytes", L.total);
    pty_plan* p = new (std::nothrow) pty_plan();
    if (!p) return fail(nullptr, PTY_ERR_INVALID_ARG, "out of host memory");
    p->d = *dims; p->L = L; p->ws = static_cast<unsigned char*>(workspace); p->device = device;
    p->last_stream = nullptr; p->launches = 0; p->fwd_valid = false; p->profiling = false; p->tm_obj_ptr = nullptr;
    p->loss_cfg = pty_loss{0, 1.f, 0.f, 0.f, 0.f, 1e-6f}; p->sparse_ready = false;
    int prev_device = -1;
    cudaError_t e = cudaGetDevice(&prev_device);
    if (e == cudaSuccess) e = cudaSetDevice(device);
    cudaDeviceProp prop{};
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, device);
    if (e == cudaSuccess && !(prop.major == 10 && prop.minor == 0)) {
        delete p;
        cudaSetDevice(prev_device);
        return fail(nullptr, PTY_ERR_UNSUPPORTED, "device %d is sm_%d%d; this library holds sm_100a code only", device, prop.major, prop.minor);
    }
    if (e == cudaSuccess && dims->N == 64) e = set_smem_attrs<Shape<64>>();
    if (e == cudaSuccess && dims->N == 256) e = set_smem_attrs<Shape<256>>();
    if (e == cudaSuccess && dims->N == 128) {
        e = cudaFuncSetAttribute(pty_fwd128g2_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G2Smem::bytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pty_fwd128g2_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G2Smem::bytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pty_fwd128g2_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G2Ring::bytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pty_fwd128g2_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G2Ring::bytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pty_bwd128g2_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G2Smem::bytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pty_bwd128g2_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G2Pair::bytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pty_bwd128g2_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G2Pair::bytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pty_bwd128g2_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G2Smem::bytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pty_probe_hat128_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F128::smem_bytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(pty_probe_grad128_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F128::smem_bytes);
    }
    if (e == cudaSuccess) e = cudaMemset(p->ws + L.scalars, 0, 256);
    if (e == cudaSuccess && (p->d.flags & PTY_FLAG_HOST)) {
        e = cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_in, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_meas, cudaEventDisableTiming);
    }
    if (prev_device >= 0 && prev_device != device) cudaSetDevice(prev_device);   // leave the caller's device as it was
    if (e != cudaSuccess) {
        delete p;
        return fail(nullptr, PTY_ERR_CUDA, "pty_create: %s", cudaGetErrorString(e));
    }
    p->num_sms = prop.multiProcessorCount;
    *out_plan = p;
    return PTY_OK;
}

static void drop_timers(pty_plan* p) {
    for (auto& t : p->timed) { cudaEventDestroy(t.a); cudaEventDestroy(t.b); }
    p->timed.clear();
}

int pty_destroy(pty_plan* plan) {
    if (plan) {
        drop_timers(plan);
        DeviceGuard dg(plan->device);
        if (plan->ev_in) cudaEventDestroy(plan->ev_in);
        if (plan->ev_meas) cudaEventDestroy(plan->ev_meas);
        if (plan->copy_stream) cudaStreamDestroy(plan->copy_stream);
    }
    delete plan;
    return PTY_OK;
}

int pty_profile(pty_plan* plan, int32_t enable) {
    if (!plan) return PTY_ERR_INVALID_ARG;
    plan->profiling = enable != 0;
    if (!enable) drop_timers(plan);
    return PTY_OK;
}

int pty_profile_read(pty_plan* plan, float* fwd_ms, int32_t* fwd_launches, float* bwd_ms, int32_t* bwd_launches) {
    if (!plan) return PTY_ERR_INVALID_ARG;
    DeviceGuard dg(plan->device);
    PTY_CUDA(plan, cudaStreamSynchronize(plan->last_stream));
    float ms[2] = {0.f, 0.f};
    int32_t n[2] = {0, 0};
    for (auto& t : plan->timed) {
        float e = 0.f;
        PTY_CUDA(plan, cudaEventElapsedTime(&e, t.a, t.b));
        ms[t.which] += e;
        n[t.which]++;
    }
    drop_timers(plan);
    if (fwd_ms) *fwd_ms = ms[0];
    if (fwd_launches) *fwd_launches = n[0];
    if (bwd_ms) *bwd_ms = ms[1];
    if (bwd_launches) *bwd_launches = n[1];
    return PTY_OK;
}

int pty_forward_loss(pty_plan* plan, const void* object, const void* probe, const float* positions, const float* tilt,
                     const float* meas_amp, int32_t B, double* loss, float* loss_per_pos, float* intensity, void* stream) {
    int rc = check_batch(plan, object, probe, positions, tilt, meas_amp, B);
    if (rc != PTY_OK) return rc;
    DeviceGuard dg(plan->device);
    if (!loss) return fail(plan, PTY_ERR_INVALID_ARG, "loss is null");
    return run_forward(plan, object, probe, positions, tilt, meas_amp, B, loss, loss_per_pos, intensity,
                       static_cast<cudaStream_t>(stream));
}

int pty_backward(pty_plan* plan, const void* object, const void* probe, const float* positions, const float* tilt,
                 const float* meas_amp, int32_t B, void* g_object, void* g_probe, float* g_positions, float* g_tilt,
                 float* g_dz, int32_t flags, void* stream) {
    int rc = check_batch(plan, object, probe, positions, tilt, meas_amp, B);
    if (rc != PTY_OK) return rc;
    DeviceGuard dg(plan->device);
    if (!g_object) return fail(plan, PTY_ERR_INVALID_ARG, "g_object is null");
    if (g_dz && plan->d.Nz > 1 && !save_hat_of(plan->d))
        return fail(plan, PTY_ERR_INVALID_ARG, "g_dz needs tilt_mode != 0 or PTY_FLAG_SPECTRA");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // The saved waves are reused only when the caller says so (PTY_BWD_REUSE_FORWARD: "nothing changed since my
    // pty_forward_loss") AND the plan has seen no other call since that forward with these very pointers.
    const bool reuse = (flags & PTY_BWD_REUSE_FORWARD) && plan->fwd_valid && plan->f_object == object &&
                       plan->f_probe == probe && plan->f_positions == positions && plan->f_tilt == tilt &&
                       plan->f_meas == meas_amp && plan->f_B == B && plan->last_stream == st;
    if (!reuse) {
        rc = run_forward(plan, object, probe, positions, tilt, meas_amp, B, plan->d_loss(), nullptr, nullptr, st);
        if (rc != PTY_OK) return rc;
    }
    return run_backward(plan, object, positions, tilt, meas_amp, B, g_object, g_probe, g_positions, g_tilt, g_dz,
                        (flags & PTY_BWD_ACCUMULATE) ? 1 : 0, st);
}

int pty_adam_update(pty_plan* plan, float* theta, const float* grad, float* m, float* v, size_t n, float lr,
                    float beta1, float beta2, float eps, int32_t t, void* stream) {
    if (!plan) return PTY_ERR_INVALID_ARG;
    DeviceGuard dg(plan->device);
    plan->last_stream = static_cast<cudaStream_t>(stream);
    plan->fwd_valid = false;            // theta may be one of the arrays the last forward read
    return adam_launch(plan, theta, grad, m, v, n, lr, beta1, beta2, eps, t, static_cast<cudaStream_t>(stream));
}

int pty_step(pty_plan* plan, void* object, void* probe, float* positions, float* tilt, const float* meas_amp,
             int32_t B, const pty_adam* hp, const pty_adam_state* s, double* loss, void* stream) {
    int rc = check_batch(plan, object, probe, positions, tilt, meas_amp, B);
    if (rc != PTY_OK) return rc;
    DeviceGuard dg(plan->device);
    if (!hp || !s || !loss) return fail(plan, PTY_ERR_INVALID_ARG, "hp, st or loss is null");
    if (!(plan->d.flags & PTY_FLAG_STEP)) return fail(plan, PTY_ERR_INVALID_ARG, "plan was created without PTY_FLAG_STEP");
    const pty_dims& d = plan->d;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    float2* g_object = plan->at<float2>(plan->L.g_object);
    float2* g_probe = plan->at<float2>(plan->L.g_probe);
    float* g_pos = plan->at<float>(plan->L.g_pos);
    float* g_tilt = plan->at<float>(plan->L.g_tilt);
    rc = run_forward(plan, object, probe, positions, tilt, meas_amp, B, loss, nullptr, nullptr, st);
    if (rc != PTY_OK) return rc;
    const bool tilt_on = d.tilt_mode != 0 && hp->lr_tilt != 0.f;
    rc = run_backward(plan, object, positions, tilt, meas_amp, B, g_object, hp->lr_probe != 0.f ? g_probe : nullptr,
                      hp->lr_positions != 0.f ? g_pos : nullptr, tilt_on ? g_tilt : nullptr, nullptr, 0, st);
    if (rc != PTY_OK) return rc;
    plan->fwd_valid = false;   // the parameters change below
    const size_t NN = (size_t)d.N * d.N;
    if ((rc = adam_launch(plan, (float*)object, (const float*)g_object, s->m_object, s->v_object,
                          plan->object_elems() * 2, hp->lr_object, hp->beta1, hp->beta2, hp->eps, hp->t, st))) return rc;
    if ((rc = adam_launch(plan, (float*)probe, (const float*)g_probe, s->m_probe, s->v_probe, (size_t)d.M * NN * 2,
                          hp->lr_probe, hp->beta1, hp->beta2, hp->eps, hp->t, st))) return rc;
    if ((rc = adam_launch(plan, positions, g_pos, s->m_positions, s->v_positions, (size_t)B * 2, hp->lr_positions,
                          hp->beta1, hp->beta2, hp->eps, hp->t, st))) return rc;
    if (tilt_on)
        if ((rc = adam_launch(plan, tilt, g_tilt, s->m_tilt, s->v_tilt, d.tilt_mode == 2 ? (size_t)B * 2 : 2, hp->lr_tilt,
                              hp->beta1, hp->beta2, hp->eps, hp->t, st))) return rc;
    return PTY_OK;
}

static int grad_host_impl(pty_plan* plan, const void* h_object, const void* h_probe, const float* h_positions,
                          const float* h_tilt, const float* h_meas_amp, int32_t B, double* h_loss, void* h_g_object,
                          void* h_g_probe, float* h_g_positions, float* h_g_tilt, void* stream, bool wait) {
    int rc = check_batch(plan, h_object, h_probe, h_positions, h_tilt, h_meas_amp, B);
    if (rc != PTY_OK) return rc;
    DeviceGuard dg(plan->device);
    if (!(plan->d.flags & PTY_FLAG_HOST)) return fail(plan, PTY_ERR_INVALID_ARG, "plan was created without PTY_FLAG_HOST");
    const pty_dims& d = plan->d;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t NN = (size_t)d.N * d.N, obj_bytes = plan->object_elems() * 8, probe_bytes = (size_t)d.M * NN * 8;
    const size_t tilt_n = d.tilt_mode == 2 ? (size_t)B * 2 : 2;
    float2* dobj = plan->at<float2>(plan->L.h_object);
    float2* dprobe = plan->at<float2>(plan->L.h_probe);
    float* dpos = plan->at<float>(plan->L.h_pos);
    float* dtilt = d.tilt_mode ? plan->at<float>(plan->L.h_tilt) : nullptr;
    float* dmeas = plan->at<float>(plan->L.h_meas);
    PTY_CUDA(plan, cudaMemcpyAsync(dobj, h_object, obj_bytes, cudaMemcpyHostToDevice, st));
    PTY_CUDA(plan, cudaMemcpyAsync(dprobe, h_probe, probe_bytes, cudaMemcpyHostToDevice, st));
    if (B) PTY_CUDA(plan, cudaMemcpyAsync(dpos, h_positions, (size_t)B * 8, cudaMemcpyHostToDevice, st));
    if (dtilt) PTY_CUDA(plan, cudaMemcpyAsync(dtilt, h_tilt, tilt_n * 4, cudaMemcpyHostToDevice, st));
    if (B) {   // measurements on the copy stream, behind whatever `st` holds so far; joined before the loss kernel
        PTY_CUDA(plan, cudaEventRecord(plan->ev_in, st));
        PTY_CUDA(plan, cudaStreamWaitEvent(plan->copy_stream, plan->ev_in, 0));
        PTY_CUDA(plan, cudaMemcpyAsync(dmeas, h_meas_amp, (size_t)B * NN * 4, cudaMemcpyHostToDevice, plan->copy_stream));
        PTY_CUDA(plan, cudaEventRecord(plan->ev_meas, plan->copy_stream));
        plan->wait_meas = true;
    }
    rc = run_forward(plan, dobj, dprobe, dpos, dtilt, dmeas, B, plan->d_loss(), nullptr, nullptr, st);
    if (rc != PTY_OK) return rc;
    float2* g_object = plan->at<float2>(plan->L.g_object);
    float2* g_probe = plan->at<float2>(plan->L.g_probe);
    float* g_pos = plan->at<float>(plan->L.g_pos);
    float* g_tilt = plan->at<float>(plan->L.g_tilt);
    rc = run_backward(plan, dobj, dpos, dtilt, dmeas, B, g_object, h_g_probe ? g_probe : nullptr,
                      h_g_positions ? g_pos : nullptr, (h_g_tilt && dtilt) ? g_tilt : nullptr, nullptr, 0, st);
    if (rc != PTY_OK) return rc;
    if (h_loss) PTY_CUDA(plan, cudaMemcpyAsync(h_loss, plan->d_loss(), 8, cudaMemcpyDeviceToHost, st));
    if (h_g_object) PTY_CUDA(plan, cudaMemcpyAsync(h_g_object, g_object, obj_bytes, cudaMemcpyDeviceToHost, st));
    if (h_g_probe) PTY_CUDA(plan, cudaMemcpyAsync(h_g_probe, g_probe, probe_bytes, cudaMemcpyDeviceToHost, st));
    if (h_g_positions && B) PTY_CUDA(plan, cudaMemcpyAsync(h_g_positions, g_pos, (size_t)B * 8, cudaMemcpyDeviceToHost, st));
    if (h_g_tilt && dtilt) PTY_CUDA(plan, cudaMemcpyAsync(h_g_tilt, g_tilt, tilt_n * 4, cudaMemcpyDeviceToHost, st));
    if (wait) PTY_CUDA(plan, cudaStreamSynchronize(st));
    return PTY_OK;
}

int pty_grad_host(pty_plan* plan, const void* h_object, const void* h_probe, const float* h_positions,
                  const float* h_tilt, const float* h_meas_amp, int32_t B, double* h_loss, void* h_g_object,
                  void* h_g_probe, float* h_g_positions, float* h_g_tilt, void* stream) {
    return grad_host_impl(plan, h_object, h_probe, h_positions, h_tilt, h_meas_amp, B, h_loss, h_g_object, h_g_probe,
                          h_g_positions, h_g_tilt, stream, true);
}

int pty_grad_host_async(pty_plan* plan, const void* h_object, const void* h_probe, const float* h_positions,
                        const float* h_tilt, const float* h_meas_amp, int32_t B, double* h_loss, void* h_g_object,
                        void* h_g_probe, float* h_g_positions, float* h_g_tilt, void* stream) {
    return grad_host_impl(plan, h_object, h_probe, h_positions, h_tilt, h_meas_amp, B, h_loss, h_g_object, h_g_probe,
                          h_g_positions, h_g_tilt, stream, false);
}

int pty_grad_host_wait(pty_plan* plan) {
    if (!plan) return PTY_ERR_INVALID_ARG;
    DeviceGuard dg(plan->device);
    PTY_CUDA(plan, cudaStreamSynchronize(plan->last_stream));
    return PTY_OK;
}


// ---------------------------------------------------------------------------- loss family (NEXT-2)
int pty_set_loss(pty_plan* plan, const pty_loss* cfg) {
    if (!plan) return PTY_ERR_INVALID_ARG;
    if (!cfg) { plan->loss_cfg = pty_loss{0, 1.f, 0.f, 0.f, 0.f, 1e-6f}; plan->fwd_valid = false; return PTY_OK; }
    if (cfg->mode != 0 && cfg->mode != 1) return fail(plan, PTY_ERR_INVALID_ARG, "loss mode must be 0 or 1");
    if (cfg->mode == 1 && !(cfg->eps > 0.f)) return fail(plan, PTY_ERR_INVALID_ARG, "Poisson eps must be > 0");
    plan->loss_cfg = *cfg;
    plan->fwd_valid = false;
    return PTY_OK;
}

int pty_loss_terms(pty_plan* plan, double* terms4) {
    if (!plan || !terms4) return PTY_ERR_INVALID_ARG;
    DeviceGuard dg(plan->device);
    PTY_CUDA(plan, cudaStreamSynchronize(plan->last_stream));
    PTY_CUDA(plan, cudaMemcpy(terms4, plan->d_stats() + ST_LG, 4 * sizeof(double), cudaMemcpyDeviceToHost));
    return PTY_OK;
}

// ---------------------------------------------------------------------------- amplitude / phase object (NEXT-2)
namespace {
int grid_for(const pty_plan* p, size_t n) {
    size_t blocks = (n + 255) / 256;
    const size_t cap = (size_t)p->num_sms * 16;
    return (int)(blocks < 1 ? 1 : blocks > cap ? cap : blocks);
}

int check_ap(pty_plan* p, const float* amp, const float* phase) {
    if (!p) return PTY_ERR_INVALID_ARG;
    if (!(p->d.flags & PTY_FLAG_AMP_PHASE)) return fail(p, PTY_ERR_INVALID_ARG, "plan was created without PTY_FLAG_AMP_PHASE");
    if (!amp || !phase) return fail(p, PTY_ERR_INVALID_ARG, "amp or phase is null");
    return PTY_OK;
}

// compose O = A exp(i phi), the coverage map of the minibatch and (loss mode 1) the sparsity term Eq. 8
int ap_prepare(pty_plan* p, const float* amp, const float* phase, const float* positions, int32_t B, cudaStream_t st) {
    const pty_dims& d = p->d;
    const size_t n = p->object_elems(), HW = (size_t)d.H * d.W;
    float2* obj = p->at<float2>(p->L.ap_object);
    float* cnt = p->at<float>(p->L.ap_cnt);
    PTY_CUDA(p, launch(p, pty_compose_object_kernel, grid_for(p, n), 256, 0, 1, st, amp, phase, obj, n));
    const bool sparse = p->loss_cfg.mode == 1 && p->loss_cfg.w_sparse != 0.f;
    if (p->loss_cfg.mode == 1) PTY_CUDA(p, cudaMemsetAsync(p->d_stats(), 0, ST_COUNT * sizeof(double), st));
    if (sparse && B) {
        PTY_CUDA(p, cudaMemsetAsync(cnt, 0, HW * sizeof(float), st));
        PTY_CUDA(p, launch(p, pty_coverage_kernel, B, 256, 0, 1, st, positions, (int)d.N, (int)d.H, (int)d.W, cnt));
        PTY_CUDA(p, launch(p, pty_sparse_sum_kernel, grid_for(p, n), 256, 0, 1, st, phase, (const float*)cnt, n, HW, p->d_stats()));
        const double n_patch = (double)B * p->n_obj() * d.Nz * d.N * d.N;
        PTY_CUDA(p, launch(p, pty_sparse_finalize_kernel, 1, 1, 0, 1, st, p->d_stats(), n_patch));
    }
    p->sparse_ready = p->loss_cfg.mode == 1;
    return PTY_OK;
}

int ap_gradients(pty_plan* p, const float* amp, const float* phase, int32_t B, float* g_amp, float* g_phase,
                 int accumulate, cudaStream_t st) {
    const pty_dims& d = p->d;
    const size_t n = p->object_elems(), HW = (size_t)d.H * d.W;
    const bool sparse = p->loss_cfg.mode == 1 && p->loss_cfg.w_sparse != 0.f && B > 0;
    const float c_sparse = sparse ? (float)((double)p->loss_cfg.w_sparse / ((double)B * p->n_obj() * d.Nz * d.N * d.N)) : 0.f;
    PTY_CUDA(p, launch(p, pty_amp_phase_grad_kernel, grid_for(p, n), 256, 0, 1, st, (const float2*)p->at<float2>(p->L.ap_g_object),
                       amp, phase, (const float*)p->at<float>(p->L.ap_cnt), c_sparse, n, HW, g_amp, g_phase, accumulate));
    return PTY_OK;
}
}  // namespace

int pty_forward_loss_ap(pty_plan* plan, const float* amp, const float* phase, const void* probe, const float* positions,
                        const float* tilt, const float* meas_amp, int32_t B, double* loss, float* loss_per_pos,
                        float* intensity, void* stream) {
    int rc = check_ap(plan, amp, phase);
    if (rc != PTY_OK) return rc;
    float2* obj = plan->at<float2>(plan->L.ap_object);
    rc = check_batch(plan, obj, probe, positions, tilt, meas_amp, B);
    if (rc != PTY_OK) return rc;
    if (!loss) return fail(plan, PTY_ERR_INVALID_ARG, "loss is null");
    DeviceGuard dg(plan->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if ((rc = ap_prepare(plan, amp, phase, positions, B, st))) return rc;
    rc = run_forward(plan, obj, probe, positions, tilt, meas_amp, B, loss, loss_per_pos, intensity, st);
    plan->fwd_valid = false;       // the composed object is private: pty_backward_ap always runs its own forward
    return rc;
}

int pty_backward_ap(pty_plan* plan, const float* amp, const float* phase, const void* probe, const float* positions,
                    const float* tilt, const float* meas_amp, int32_t B, float* g_amp, float* g_phase, void* g_probe,
                    float* g_positions, float* g_tilt, float* g_dz, int32_t flags, void* stream) {
    int rc = check_ap(plan, amp, phase);
    if (rc != PTY_OK) return rc;
    float2* obj = plan->at<float2>(plan->L.ap_object);
    rc = check_batch(plan, obj, probe, positions, tilt, meas_amp, B);
    if (rc != PTY_OK) return rc;
    if (!g_amp || !g_phase) return fail(plan, PTY_ERR_INVALID_ARG, "g_amp or g_phase is null");
    if (g_dz && plan->d.Nz > 1 && !save_hat_of(plan->d))
        return fail(plan, PTY_ERR_INVALID_ARG, "g_dz needs tilt_mode != 0 or PTY_FLAG_SPECTRA");
    DeviceGuard dg(plan->device);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if ((rc = ap_prepare(plan, amp, phase, positions, B, st))) return rc;
    if ((rc = run_forward(plan, obj, probe, positions, tilt, meas_amp, B, plan->d_loss(), nullptr, nullptr, st))) return rc;
    plan->fwd_valid = false;
    const int acc = (flags & PTY_BWD_ACCUMULATE) ? 1 : 0;
    // the complex gradient of THIS minibatch goes to the workspace (never accumulated there); amp / phase accumulate
    if ((rc = run_backward(plan, obj, positions, tilt, meas_amp, B, plan->at<float2>(plan->L.ap_g_object), g_probe,
                           g_positions, g_tilt, g_dz, acc, st, 0))) return rc;
    return ap_gradients(plan, amp, phase, B, g_amp, g_phase, acc, st);
}

int pty_step_ap(pty_plan* plan, float* amp, float* phase, void* probe, float* positions, float* tilt, const float* meas_amp,
                int32_t B, const pty_adam_ap* hp, const pty_adam_state_ap* s, double* loss, void* stream) {
    int rc = check_ap(plan, amp, phase);
    if (rc != PTY_OK) return rc;
    float2* obj = plan->at<float2>(plan->L.ap_object);
    rc = check_batch(plan, obj, probe, positions, tilt, meas_amp, B);
    if (rc != PTY_OK) return rc;
    if (!hp || !s || !loss) return fail(plan, PTY_ERR_INVALID_ARG, "hp, st or loss is null");
    if (!(plan->d.flags & PTY_FLAG_STEP)) return fail(plan, PTY_ERR_INVALID_ARG, "plan was created without PTY_FLAG_STEP");
    DeviceGuard dg(plan->device);
    const pty_dims& d = plan->d;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // the step's real gradient buffers: g_amp and g_phase share the STEP buffer reserved for a complex g_object
    float* g_amp = plan->at<float>(plan->L.g_object);
    float* g_phase = g_amp + plan->object_elems();
    float2* g_probe = plan->at<float2>(plan->L.g_probe);
    float* g_pos = plan->at<float>(plan->L.g_pos);
    float* g_tilt = plan->at<float>(plan->L.g_tilt);
    if ((rc = ap_prepare(plan, amp, phase, positions, B, st))) return rc;
    if ((rc = run_forward(plan, obj, probe, positions, tilt, meas_amp, B, loss, nullptr, nullptr, st))) return rc;
    const bool tilt_on = d.tilt_mode != 0 && hp->lr_tilt != 0.f;
    if ((rc = run_backward(plan, obj, positions, tilt, meas_amp, B, plan->at<float2>(plan->L.ap_g_object),
                           hp->lr_probe != 0.f ? g_probe : nullptr, hp->lr_positions != 0.f ? g_pos : nullptr,
                           tilt_on ? g_tilt : nullptr, nullptr, 0, st))) return rc;
    plan->fwd_valid = false;
    if ((rc = ap_gradients(plan, amp, phase, B, g_amp, g_phase, 0, st))) return rc;
    const size_t NN = (size_t)d.N * d.N, n = plan->object_elems();
    if ((rc = adam_launch(plan, amp, g_amp, s->m_amp, s->v_amp, n, hp->lr_amp, hp->beta1, hp->beta2, hp->eps, hp->t, st))) return rc;
    if ((rc = adam_launch(plan, phase, g_phase, s->m_phase, s->v_phase, n, hp->lr_phase, hp->beta1, hp->beta2, hp->eps, hp->t, st))) return rc;
    if ((rc = adam_launch(plan, (float*)probe, (const float*)g_probe, s->m_probe, s->v_probe, (size_t)d.M * NN * 2,
                          hp->lr_probe, hp->beta1, hp->beta2, hp->eps, hp->t, st))) return rc;
    if ((rc = adam_launch(plan, positions, g_pos, s->m_positions, s->v_positions, (size_t)B * 2, hp->lr_positions,
                          hp->beta1, hp->beta2, hp->eps, hp->t, st))) return rc;
    if (tilt_on)
        if ((rc = adam_launch(plan, tilt, g_tilt, s->m_tilt, s->v_tilt, d.tilt_mode == 2 ? (size_t)B * 2 : 2, hp->lr_tilt,
                              hp->beta1, hp->beta2, hp->eps, hp->t, st))) return rc;
    return PTY_OK;
}

// ---------------------------------------------------------------------------- constraints (NEXT-3)
namespace {
// Eq. 13 on a float array viewed as [outer][Nz][plane]
int rz_filter_launch(pty_plan* p, float* x, size_t outer, size_t plane, float sigma_z, cudaStream_t st) {
    const int Nz = p->d.Nz;
    if (!(sigma_z > 0.f) || Nz < 2) return PTY_OK;
    const int R = std::max(1, (int)std::ceil(2.0 * (double)sigma_z));
    if (R > 8) return fail(p, PTY_ERR_UNSUPPORTED, "r_z filter: sigma_z = %g needs a radius of %d slices (max 8)", (double)sigma_z, R);
    RzTaps taps{};           // by value into the launch: nothing on the host has to outlive this call (stream capture)
    double sum = 0.0;
    for (int j = -R; j <= R; ++j) sum += std::exp(-(double)j * j / (2.0 * (double)sigma_z * sigma_z));
    for (int j = -R; j <= R; ++j) taps.t[j + R] = (float)(std::exp(-(double)j * j / (2.0 * (double)sigma_z * sigma_z)) / sum);
    const size_t columns = outer * plane;
    const int grid = grid_for(p, columns);
    cudaError_t e = cudaSuccess;
    switch (R) {
#define PTY_RZ(RR) case RR: e = launch(p, pty_rz_filter_kernel<RR>, grid, 256, 0, 1, st, x, Nz, plane, columns, taps); break;
        PTY_RZ(1) PTY_RZ(2) PTY_RZ(3) PTY_RZ(4) PTY_RZ(5) PTY_RZ(6) PTY_RZ(7) PTY_RZ(8)
#undef PTY_RZ
    }
    PTY_CUDA(p, e);
    return PTY_OK;
}
}  // namespace

int pty_constrain(pty_plan* plan, float* amp, float* phase, void* probe, const pty_constraints* c, void* stream) {
    if (!plan) return PTY_ERR_INVALID_ARG;
    if (!c) return fail(plan, PTY_ERR_INVALID_ARG, "constraints is null");
    DeviceGuard dg(plan->device);
    const pty_dims& d = plan->d;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    plan->last_stream = st;
    plan->fwd_valid = false;
    int rc;
    const size_t n = plan->object_elems(), HW = (size_t)d.H * d.W;
    if (c->sigma_z > 0.f) {
        if (amp && (rc = rz_filter_launch(plan, amp, (size_t)plan->n_obj(), HW, c->sigma_z, st))) return rc;
        if (phase && (rc = rz_filter_launch(plan, phase, (size_t)plan->n_obj(), HW, c->sigma_z, st))) return rc;
    }
    const int pos = c->phase_positive && phase, clamp = c->clamp_amp && amp;
    if (clamp && !(c->amp_min <= c->amp_max)) return fail(plan, PTY_ERR_INVALID_ARG, "amp_min > amp_max");
    if (pos || clamp)
        PTY_CUDA(plan, launch(plan, pty_clip_clamp_kernel, grid_for(plan, n), 256, 0, 1, st, amp, phase, n, pos, clamp, c->amp_min, c->amp_max));
    if (c->ortho_probe) {
        if (!probe) return fail(plan, PTY_ERR_INVALID_ARG, "ortho_probe needs the probe");
        if (d.M > kMaxModes) return fail(plan, PTY_ERR_UNSUPPORTED, "probe orthogonalisation supports M <= %d", kMaxModes);
        const size_t NN = (size_t)d.N * d.N;
        double2* G = plan->at<double2>(plan->L.gram);
        double2* V = plan->at<double2>(plan->L.eigv);
        double* lam = plan->at<double>(plan->L.eigl);
        PTY_CUDA(plan, launch(plan, pty_gram_kernel, d.M * (d.M + 1) / 2, 256, 0, 1, st, (const float2*)probe, (int)d.M, NN, G));
        PTY_CUDA(plan, launch(plan, pty_eigh_kernel, 1, 32, 0, 1, st, (const double2*)G, (int)d.M, V, lam));
        PTY_CUDA(plan, launch(plan, pty_mix_modes_kernel, grid_for(plan, NN), 256, 0, 1, st, (float2*)probe, (int)d.M, NN, (const double2*)V));
    }
    return PTY_OK;
}

int pty_rz_filter_object(pty_plan* plan, void* object, float sigma_z, void* stream) {
    if (!plan) return PTY_ERR_INVALID_ARG;
    if (!object) return fail(plan, PTY_ERR_INVALID_ARG, "object is null");
    DeviceGuard dg(plan->device);
    plan->last_stream = static_cast<cudaStream_t>(stream);
    plan->fwd_valid = false;
    // complex64 = interleaved (re, im): a plane of H W complex values is 2 H W floats
    return rz_filter_launch(plan, static_cast<float*>(object), (size_t)plan->n_obj(), (size_t)plan->d.H * plan->d.W * 2, sigma_z,
                            static_cast<cudaStream_t>(stream));
}

// Probe-mode orthogonalisation without a plan, a workspace or any allocation (include/pty.h): the three kernels of
// pty_constrain's ortho_probe branch, with their scratch in the library's own static device array.
int pty_ortho_probe_noalloc(void* probe, int32_t M, int32_t N, int device, void* stream) {
    if (!probe) return fail(nullptr, PTY_ERR_INVALID_ARG, "pty_ortho_probe_noalloc: probe is null");
    if (reinterpret_cast<uintptr_t>(probe) % 8) return fail(nullptr, PTY_ERR_INVALID_ARG, "pty_ortho_probe_noalloc: probe must be 8-byte aligned");
    if (M < 1) return fail(nullptr, PTY_ERR_INVALID_ARG, "pty_ortho_probe_noalloc: M = %d, need at least one mode", (int)M);
    if (M > PTY_ORTHO_NOALLOC_MAX_MODES)
        return fail(nullptr, PTY_ERR_UNSUPPORTED, "pty_ortho_probe_noalloc: M = %d modes do not fit the fixed %d-byte scratch (limit: %d modes)",
                    (int)M, (int)PTY_ORTHO_NOALLOC_SCRATCH_BYTES, (int)PTY_ORTHO_NOALLOC_MAX_MODES);
    if (N < 1 || N > 4096) return fail(nullptr, PTY_ERR_INVALID_ARG, "pty_ortho_probe_noalloc: N = %d, need 1 <= N <= 4096", (int)N);
    if (device < 0 || device >= kNoAllocMaxDevices)
        return fail(nullptr, PTY_ERR_INVALID_ARG, "pty_ortho_probe_noalloc: device %d outside [0, %d)", device, kNoAllocMaxDevices);
    DeviceGuard dg(device);
    int current = -1;
    PTY_CUDA(nullptr, cudaGetDevice(&current));
    if (current != device) return fail(nullptr, PTY_ERR_INVALID_ARG, "pty_ortho_probe_noalloc: cannot make device %d current", device);
    unsigned char* scratch = nullptr;
    int rc;
    if ((rc = noalloc_scratch(device, &scratch))) return rc;
    // the workspace layout of the plan path (make_layout: gram, eigv, eigl), at its largest M
    constexpr size_t kMat = (size_t)PTY_ORTHO_NOALLOC_MAX_MODES * PTY_ORTHO_NOALLOC_MAX_MODES * sizeof(double2);
    double2* G = reinterpret_cast<double2*>(scratch);
    double2* V = reinterpret_cast<double2*>(scratch + kMat);
    double* lam = reinterpret_cast<double*>(scratch + 2 * kMat);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t NN = (size_t)N * N;
    const size_t blocks = std::min<size_t>((NN + 255) / 256, 148 * 16);
    // every G, V, lam element read below is written first by the kernel before it: nothing needs clearing between calls
    pty_gram_kernel<<<M * (M + 1) / 2, 256, 0, st>>>((const float2*)probe, (int)M, NN, G);
    PTY_CUDA(nullptr, cudaGetLastError());
    pty_eigh_kernel<<<1, 32, 0, st>>>((const double2*)G, (int)M, V, lam);
    PTY_CUDA(nullptr, cudaGetLastError());
    pty_mix_modes_kernel<<<(unsigned)blocks, 256, 0, st>>>((float2*)probe, (int)M, NN, (const double2*)V);
    PTY_CUDA(nullptr, cudaGetLastError());
    return PTY_OK;
}

int pty_status(pty_plan* plan, int32_t* device_flags) {
    if (!plan) return PTY_ERR_INVALID_ARG;
    DeviceGuard dg(plan->device);
    PTY_CUDA(plan, cudaStreamSynchronize(plan->last_stream));
    int flags = 0;
    PTY_CUDA(plan, cudaMemcpy(&flags, plan->d_flags(), sizeof(int), cudaMemcpyDeviceToHost));
    PTY_CUDA(plan, cudaMemset(plan->d_flags(), 0, sizeof(int)));
    if (device_flags) *device_flags = flags;
    PTY_CUDA(plan, cudaGetLastError());
    if (flags & 1) return fail(plan, PTY_ERR_BOUNDS, "a scan position's crop left the object and was clamped");
    if (flags & 2) return fail(plan, PTY_ERR_ZERO_DATA, "loss mode 1 on a minibatch of all-zero measurements: the normalised terms were set to 0");
    return PTY_OK;
}

int64_t pty_launch_count(const pty_plan* plan) { return plan ? plan->launches : 0; }

const char* pty_last_error(const pty_plan* plan) { return plan ? plan->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
