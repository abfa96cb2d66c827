// pty_fft.cuh -- register butterflies and the shared-memory line-FFT passes.
//
// A wave of N x N complex64 lives in shared memory as S[N][PITCH] (PITCH odd).  One "pass" is a
// 1-D FFT over the SLOW index (rows) for every line (column), done in two register stages
// (N = R1*R2, decimation in time) and written back TRANSPOSED, so that the next pass again
// transforms over the slow index.  Two passes = one 2-D FFT, and the wave is back in (y, x)
// orientation.  Lanes of a warp always run along the line index: shared-memory reads are
// lane-contiguous, transposed writes hit stride PITCH (odd) -> conflict-free for 8-byte words.
// For N = 256 the N lines are split over a cluster of CL = 4 CTAs (64 lines each); the
// transposed write then goes to the owning CTA's shared memory through DSMEM.
//
//   X[k1 + R1 k2] = sum_{n2} W_N^{n2 k1} W_{R2}^{n2 k2} [ sum_{n1} x[R2 n1 + n2] W_{R1}^{n1 k1} ]
//
// DIR = -1: forward kernel exp(-2 pi i nk/N);  DIR = +1: inverse (unscaled).
#pragma once
#ifndef PTY_PORT_INCLUDED
#include "pty_port.cuh"
#endif

#ifndef PTY_CLUSTER_RELAXED
#define PTY_CLUSTER_RELAXED 1   // N = 256: the write-after-read cluster barrier of stage B arrives without a release fence (c5: 22.9 -> 22.2 ms)
#endif

namespace pty {

// ----------------------------------------------------------------------------- complex helpers
// Packed FP32x2 arithmetic (FADD2 / FMUL2 / FFMA2 on sm_100a): a complex value is one 64-bit register
// pair, and the operand modifiers of the packed instructions (half swap, per-half negate, scalar
// broadcast) absorb the swaps and sign changes, so every complex operation below is one or two
// instructions.  Same FP32 lane throughput as scalar code, half the issue slots (profiles/r03_fp32_pipe.md).
PTY_DEV float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
PTY_DEV float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
PTY_DEV float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
PTY_DEV float2 cmulc(float2 a, float2 b) { return make_float2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }
PTY_DEV float2 cscale(float2 a, float s) { return make_float2(a.x * s, a.y * s); }
PTY_DEV float2 cconj(float2 a) { return make_float2(a.x, -a.y); }
// variable twiddles of the cross-thread radix-4 stage (scalar form: the packed one measured +-0)
PTY_DEV float2 cmul_tw(float2 a, float2 w) { return make_float2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x); }
PTY_DEV float2 cmulc_tw(float2 w, float2 a) { return make_float2(w.x * a.x + w.y * a.y, w.x * a.y - w.y * a.x); }

// a * exp(DIR * i * pi/2): forward multiplies by -i, inverse by +i
template <int DIR> PTY_DEV float2 mul_qi(float2 a) {
    return DIR < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
}
// a * (c + i*DIR*s) with c, s the cos/sin of a positive angle
template <int DIR> PTY_DEV float2 mul_cs(float2 a, float c, float s) {
    const float2 t = __fmul2_rn(a, make_float2(c, c));
    return DIR < 0 ? __ffma2_rn(make_float2(a.y, a.x), make_float2(s, -s), t)
                   : __ffma2_rn(make_float2(a.y, a.x), make_float2(-s, s), t);
}

// ----------------------------------------------------------------------------- radix-4 / 8 / 16
template <int DIR> PTY_DEV void bfly4(float2& a0, float2& a1, float2& a2, float2& a3) {
    float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = mul_qi<DIR>(csub(a1, a3));
    a0 = cadd(t0, t2); a2 = csub(t0, t2); a1 = cadd(t1, t3); a3 = csub(t1, t3);
}

template <int R, int DIR> struct RegFFT;

template <int DIR> struct RegFFT<8, DIR> {
    static PTY_DEV void run(float2 (&v)[8]) {
        const float h = 0.70710678118654752440f;
        bfly4<DIR>(v[0], v[2], v[4], v[6]);           // E_k at v[0],v[2],v[4],v[6]
        bfly4<DIR>(v[1], v[3], v[5], v[7]);           // O_k at v[1],v[3],v[5],v[7]
        float2 o1 = mul_cs<DIR>(v[3], h, h);          // W8^1
        float2 o2 = mul_qi<DIR>(v[5]);                // W8^2
        float2 o3 = mul_cs<DIR>(mul_qi<DIR>(v[7]), h, h);   // W8^3 = W8^2 W8^1
        float2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6], o0 = v[1];
        v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
        v[1] = cadd(e1, o1); v[5] = csub(e1, o1);
        v[2] = cadd(e2, o2); v[6] = csub(e2, o2);
        v[3] = cadd(e3, o3); v[7] = csub(e3, o3);
    }
};

template <int DIR> struct RegFFT<16, DIR> {
    static PTY_DEV void run(float2 (&v)[16]) {
        const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;   // pi/8
        const float h = 0.70710678118654752440f;                                   // pi/4
        // stage 1: 4-point DFTs over n1 for every n2 (inputs v[4 n1 + n2]); result k1 at v[4 k1 + n2]
#pragma unroll
        for (int n2 = 0; n2 < 4; ++n2) bfly4<DIR>(v[n2], v[4 + n2], v[8 + n2], v[12 + n2]);
        // twiddles W16^{n2 k1}
        v[4 + 1] = mul_cs<DIR>(v[4 + 1], c1, s1);                  // k1=1,n2=1: W^1
        v[4 + 2] = mul_cs<DIR>(v[4 + 2], h, h);                    // W^2
        v[4 + 3] = mul_cs<DIR>(v[4 + 3], s1, c1);                  // W^3
        v[8 + 1] = mul_cs<DIR>(v[8 + 1], h, h);                    // k1=2,n2=1: W^2
        v[8 + 2] = mul_qi<DIR>(v[8 + 2]);                          // W^4
        v[8 + 3] = mul_cs<DIR>(mul_qi<DIR>(v[8 + 3]), h, h);       // W^6 = W^4 W^2
        v[12 + 1] = mul_cs<DIR>(v[12 + 1], s1, c1);                // k1=3,n2=1: W^3
        v[12 + 2] = mul_cs<DIR>(mul_qi<DIR>(v[12 + 2]), h, h);     // W^6
        v[12 + 3] = mul_cs<DIR>(mul_qi<DIR>(mul_qi<DIR>(v[12 + 3])), c1, s1);   // W^9 = W^8 W^1
        // stage 2: 4-point DFTs over n2 for every k1; X[k1 + 4 k2] lands in v[4 k1 + k2]
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) bfly4<DIR>(v[4 * k1], v[4 * k1 + 1], v[4 * k1 + 2], v[4 * k1 + 3]);
        // to natural order: out[k1 + 4 k2] = v[4 k1 + k2]  (a 4x4 transpose)
        float2 t;
        t = v[1]; v[1] = v[4]; v[4] = t;
        t = v[2]; v[2] = v[8]; v[8] = t;
        t = v[3]; v[3] = v[12]; v[12] = t;
        t = v[6]; v[6] = v[9]; v[9] = t;
        t = v[7]; v[7] = v[13]; v[13] = t;
        t = v[11]; v[11] = v[14]; v[14] = t;
    }
};

// ----------------------------------------------------------------------------- shapes
template <int N_> struct Shape;
template <> struct Shape<64>  { static constexpr int N = 64,  R1 = 8,  R2 = 8,  CL = 1, NL = 64,  NT = 256; };
template <> struct Shape<256> { static constexpr int N = 256, R1 = 16, R2 = 16, CL = 4, NL = 64,  NT = 512; };

template <class SH> struct ShapeInfo {
    static constexpr int N = SH::N, R1 = SH::R1, R2 = SH::R2, CL = SH::CL, NL = SH::NL, NT = SH::NT;
    static constexpr int PITCH = NL + 1;
    static constexpr int TA = (R2 * NL) / NT;      // stage-A tasks per thread
    static constexpr int TB = (R1 * NL) / NT;      // stage-B tasks per thread
    static constexpr int SWEEP = (N * NL) / NT;    // elements per thread in a sweep
    static_assert(R1 * R2 == N, "radix split");
    static_assert((R2 * NL) % NT == 0 && (R1 * NL) % NT == 0, "task split");
    static_assert(NL % 32 == 0, "a warp must stay inside one task group");
    static constexpr size_t wave_bytes = size_t(N) * PITCH * sizeof(float2);
    static constexpr size_t table_bytes = size_t(5) * N * sizeof(float2) + 64 * sizeof(float);
    // cluster shapes: two staging tiles NL x (NL + 1) for the coalesced DSMEM transpose (stage_b)
    static constexpr size_t stage_bytes = CL > 1 ? size_t(2) * NL * (NL + 1) * sizeof(float2) : 0;
    // cluster shapes: + the mbarrier that counts the bytes arriving from the peers (st.async exchange)
    static constexpr size_t smem_bytes = wave_bytes + table_bytes + stage_bytes + (CL > 1 ? 16 : 0);
};

// Per-CTA view: thread id, rank in the cluster, the wave buffer of every CTA of the cluster
// (Sr[rank] == S), the small tables.
template <class SH> struct Cta {
    int tid, rank;
    float2* S;
    float2* Sr[SH::CL];
    float2 *tw, *Ey, *Ex, *My, *Mx;   // [N] each: twiddles exp(-2 pi i j/N); shift and propagator factors
    float* red;                       // [64] block-reduction scratch
    float2* stg;                      // cluster shapes: 2 staging tiles [NL][NL + 1]
    unsigned long long* rx;           // cluster shapes: mbarrier completed by the peers' st.async of one exchange
    mutable unsigned rx_phase;        // parity of the exchange this CTA waits for next
};

template <class SH> PTY_DEV void sync_all() {
    if (SH::CL > 1) pty_cluster_sync(); else pty_cta_sync();
}
// Execution barrier only (write-after-read protection: every thread of the cluster has finished READING the waves into
// registers; nothing written before it has to become visible), so the arrive carries no release fence.
// This is an argument from how the hardware executes the barrier (a thread's earlier ld.shared have returned their data
// before it can arrive: the values are consumed by the register transposes in between), NOT from the PTX memory model,
// which gives a relaxed arrive no happens-before edge to the peers' later st.async.  Hence a compile-time switch
// (PTY_CLUSTER_RELAXED = 0: the fenced barrier), and tests/test_gpu_cluster_order.py compares the bits of both builds.
template <class SH> PTY_DEV void sync_all_war() {
#if PTY_CLUSTER_RELAXED
    if (SH::CL > 1) {
        asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
        asm volatile("barrier.cluster.wait.aligned;" ::: "memory");
    } else {
        pty_cta_sync();
    }
#else
    sync_all<SH>();
#endif
}

// ----------------------------------------------------------------------------- stage A
// In::load(cta, n2, line, gline, v) fills v[n1] = element (row = R2 n1 + n2, line) of the input,
// with whatever pointwise work is fused there (see pty_kernels.cuh).
template <class SH, int DIR, class In>
PTY_DEV void stage_a(const Cta<SH>& c, In& in) {
    using I = ShapeInfo<SH>;
#pragma unroll
    for (int it = 0; it < I::TA; ++it) {
        const int t = it * I::NT + c.tid;
        const int line = t % I::NL, n2 = t / I::NL;
        float2 v[I::R1];
        in.load(c, n2, line, c.rank * I::NL + line, v);
        RegFFT<I::R1, DIR>::run(v);
#pragma unroll
        for (int k1 = 1; k1 < I::R1; ++k1) {
            float2 w = c.tw[n2 * k1];
            if (DIR > 0) w.y = -w.y;
            v[k1] = cmul(v[k1], w);
        }
#pragma unroll
        for (int k1 = 0; k1 < I::R1; ++k1) c.S[(I::R2 * k1 + n2) * I::PITCH + line] = v[k1];
    }
}

// Transposed exchange of stage B for cluster shapes, CTA of rank RANK: the registers v[it][k2] with k2 / K2D == d go to
// CTA d, rows [RANK NL, +NL) of its wave.
template <class SH, int RANK>
PTY_DEV void stage_b_exchange(const Cta<SH>& c, float2 (&v)[ShapeInfo<SH>::TB][SH::R2]) {
    using I = ShapeInfo<SH>;
    static_assert(SH::CL <= 4, "switch in stage_b");
    constexpr int TP = I::NL + 1, K2D = I::NL / I::R1;          // k2 values per destination
    static_assert(I::NL % I::R1 == 0 && (I::NL * I::NL) % I::NT == 0, "tile split");
#pragma unroll
    for (int rr = 0; rr < SH::CL; ++rr) {
        const int d = (RANK + rr) % SH::CL;
        if (rr == 0) {      // own rows: scattered 8-byte stores straight into the wave (odd pitch: conflict-free)
#pragma unroll
            for (int it = 0; it < I::TB; ++it) {
                const int t = it * I::NT + c.tid;
                const int line = t % I::NL, k1 = t / I::NL;
#pragma unroll
                for (int k2 = 0; k2 < I::R2; ++k2)
                    if (k2 / K2D == d) c.S[(RANK * I::NL + line) * I::PITCH + (k1 + I::R1 * (k2 % K2D))] = v[it][k2];
            }
            continue;
        }
        float2* tile = c.stg + (rr & 1) * (I::NL * TP);
#pragma unroll
        for (int it = 0; it < I::TB; ++it) {
            const int t = it * I::NT + c.tid;
            const int line = t % I::NL, k1 = t / I::NL;
#pragma unroll
            for (int k2 = 0; k2 < I::R2; ++k2)
                if (k2 / K2D == d) tile[line * TP + (k1 + I::R1 * (k2 % K2D))] = v[it][k2];
        }
        pty_cta_sync();
        unsigned rbase;
        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rbase)
                     : "r"((unsigned)__cvta_generic_to_shared(c.S + (size_t)(RANK * I::NL) * I::PITCH)), "r"(d));
        unsigned rbar;
        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rbar) : "r"((unsigned)__cvta_generic_to_shared(c.rx)), "r"(d));
        float2 tv[(I::NL * I::NL) / I::NT];
#pragma unroll
        for (int j = 0; j < (I::NL * I::NL) / I::NT; ++j) {
            const int idx = j * I::NT + c.tid;
            tv[j] = tile[(idx / I::NL) * TP + idx % I::NL];
        }
#pragma unroll
        for (int j = 0; j < (I::NL * I::NL) / I::NT; ++j) {
            const int idx = j * I::NT + c.tid;
            const unsigned a = rbase + (unsigned)(((idx / I::NL) * I::PITCH + idx % I::NL) * sizeof(float2));
            // asynchronous remote store: its 8 bytes are counted on the RECEIVER's mbarrier, so the exchange needs neither
            // a release fence (which would also drain this thread's saved-wave stores to HBM) nor a closing cluster barrier
            asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];"
                         ::"r"(a), "f"(tv[j].x), "f"(tv[j].y), "r"(rbar) : "memory");
        }
    }
}

// ----------------------------------------------------------------------------- stage B
// Reads everything into registers, synchronises, then writes the transposed result:
// element (old line L_global, k) goes to row L_global, column k of the new orientation,
// i.e. to CTA k / NL at Sr[.][L_global * PITCH + k % NL].
template <class SH, int DIR, bool TR>
PTY_DEV void stage_b(const Cta<SH>& c) {
    using I = ShapeInfo<SH>;
    float2 v[I::TB][I::R2];
#pragma unroll
    for (int it = 0; it < I::TB; ++it) {
        const int t = it * I::NT + c.tid;
        const int line = t % I::NL, k1 = t / I::NL;
#pragma unroll
        for (int n2 = 0; n2 < I::R2; ++n2) v[it][n2] = c.S[(I::R2 * k1 + n2) * I::PITCH + line];
        RegFFT<I::R2, DIR>::run(v[it]);
    }
    if constexpr (!TR) {
        // in place: frequency k = k1 + R1 k2 of every line goes to row k of the same line -- local to the CTA, so a
        // CTA barrier on each side is all it takes (no cluster barrier, no exchange)
        pty_cta_sync();
#pragma unroll
        for (int it = 0; it < I::TB; ++it) {
            const int t = it * I::NT + c.tid;
            const int line = t % I::NL, k1 = t / I::NL;
#pragma unroll
            for (int k2 = 0; k2 < I::R2; ++k2) c.S[(k1 + I::R1 * k2) * I::PITCH + line] = v[it][k2];
        }
        pty_cta_sync();
        return;
    }
    sync_all_war<SH>();
    if constexpr (SH::CL == 1) {
#pragma unroll
        for (int it = 0; it < I::TB; ++it) {
            const int t = it * I::NT + c.tid;
            const int line = t % I::NL, k1 = t / I::NL;
#pragma unroll
            for (int k2 = 0; k2 < I::R2; ++k2) c.S[line * I::PITCH + (k1 + I::R1 * k2)] = v[it][k2];
        }
    } else {
        // The NL x NL tile that goes to CTA d is first assembled in local shared memory (scattered 8-byte stores,
        // cheap locally) and then copied to the owner with lane-contiguous stores: a warp writes 256 contiguous
        // bytes of remote shared memory instead of 32 separate 8-byte words (the scattered form ran at 10 % issue
        // utilisation, stalled on lg_throttle -- round 1).  Two tiles alternate, one CTA barrier
        // per destination; destinations start at the own rank so that the four CTAs do not target one peer.
        // The rank is a template parameter of the exchange (a CTA-uniform switch), so the destination of every register
        // is known at compile time: no predicated-off stores, and the tile for the own CTA is written in place.
        // this CTA expects the tiles of its CL - 1 peers (one arrival: this post; the bytes: their st.async)
        if (c.tid == 0) mbar_expect_tx(c.rx, (unsigned)((SH::CL - 1) * I::NL * I::NL * sizeof(float2)));
        switch (c.rank) {
            case 0: stage_b_exchange<SH, 0>(c, v); break;
            case 1: stage_b_exchange<SH, 1 % SH::CL>(c, v); break;
            case 2: stage_b_exchange<SH, 2 % SH::CL>(c, v); break;
            default: stage_b_exchange<SH, 3 % SH::CL>(c, v); break;
        }
        mbar_wait(c.rx, c.rx_phase);      // every peer's tile has landed in this CTA's wave
        c.rx_phase ^= 1u;
        pty_cta_sync();                   // ... and this CTA's own tile (written in place by its threads)
        return;
    }
    sync_all<SH>();
}

// Plain input: the wave itself.
struct InSmem {
    template <class SH, int R>
    PTY_DEV void load(const Cta<SH>& c, int n2, int line, int, float2 (&v)[R]) {
        using I = ShapeInfo<SH>;
#pragma unroll
        for (int n1 = 0; n1 < R; ++n1) v[n1] = c.S[(I::R2 * n1 + n2) * I::PITCH + line];
    }
};

// One full pass: stage A (with its fused input work), stage B, and the write-back -- transposed (TR: lines <-> rows,
// through DSMEM on cluster shapes) or in place.  A 2-D FFT is a transposing pass followed by an in-place pass: real
// space is held as [y][x line], k space TRANSPOSED as [kx][ky line]; the pointwise k-space steps and every k-space
// workspace array (P^, Psi, psi^, I, seed weights, G^_P) use that orientation, so ONE exchange per 2-D FFT suffices.
template <class SH, int DIR, bool TR, class In>
PTY_DEV void fft_pass(const Cta<SH>& c, In& in) {
    stage_a<SH, DIR>(c, in);
    pty_cta_sync();
    stage_b<SH, DIR, TR>(c);
}
// Stage B of an in-place pass, the pointwise step that follows the 2-D FFT, and stage A of the NEXT 2-D FFT's
// transposing pass, fused in registers.  All passes run over the slow index, and with R1 == R2 the frequencies a
// stage-B task (line, k1) produces, rows k1 + R1 k2, are exactly the rows R2 n1 + n2 (n1 = k2, n2 = k1) that one
// stage-A task of the next transform consumes: the values never go back to shared memory in between (one store, one
// load and one CTA barrier less per 2-D FFT).  op.apply(c, n2, line, gline, v) transforms v[n1] = element
// (row R2 n1 + n2, line) in place.  Reads (row blocks) and writes (row combs) of different tasks overlap, hence the
// barrier between them.
template <class SH, int DIRB, int DIRA, class Op>
PTY_DEV void stage_b_op_a(const Cta<SH>& c, Op& op) {
    using I = ShapeInfo<SH>;
    static_assert(I::R1 == I::R2, "fused stage B -> stage A needs a square radix split");
    float2 v[I::TB][I::R2];
#pragma unroll
    for (int it = 0; it < I::TB; ++it) {
        const int t = it * I::NT + c.tid;
        const int line = t % I::NL, k1 = t / I::NL;
#pragma unroll
        for (int n2 = 0; n2 < I::R2; ++n2) v[it][n2] = c.S[(I::R2 * k1 + n2) * I::PITCH + line];
        RegFFT<I::R2, DIRB>::run(v[it]);
        op.apply(c, k1, line, c.rank * I::NL + line, v[it]);
        RegFFT<I::R1, DIRA>::run(v[it]);
#pragma unroll
        for (int kk = 1; kk < I::R1; ++kk) {
            float2 w = c.tw[k1 * kk];
            if (DIRA > 0) w.y = -w.y;
            v[it][kk] = cmul(v[it][kk], w);
        }
    }
    pty_cta_sync();
#pragma unroll
    for (int it = 0; it < I::TB; ++it) {
        const int t = it * I::NT + c.tid;
        const int line = t % I::NL, k1 = t / I::NL;
#pragma unroll
        for (int kk = 0; kk < I::R1; ++kk) c.S[(I::R2 * kk + k1) * I::PITCH + line] = v[it][kk];
    }
}

// A chain of 2-D FFTs with pointwise steps between them:
//   fft_begin<DIR>(in)        first transform: transposing pass (inputs from `in`), stage A of the in-place pass
//   fft_link<DIRB, DIRA>(op)  finishes transform DIRB, applies `op`, runs transform DIRA up to the same point
//   fft_end<DIR>()            finishes the last transform (plain in-place stage B)
// Orientation: real [y][x] -> k space [kx][ky] (DIR < 0) and back (DIR > 0); `in` / `op` see the source side.
template <class SH, int DIR, class In>
PTY_DEV void fft_begin(const Cta<SH>& c, In& in) {
    InSmem plain;
    fft_pass<SH, DIR, true>(c, in);
    stage_a<SH, DIR>(c, plain);
    pty_cta_sync();
}
template <class SH, int DIRB, int DIRA, class Op>
PTY_DEV void fft_link(const Cta<SH>& c, Op& op) {
    InSmem plain;
    stage_b_op_a<SH, DIRB, DIRA>(c, op);
    pty_cta_sync();
    stage_b<SH, DIRA, true>(c);
    stage_a<SH, DIRA>(c, plain);
    pty_cta_sync();
}
template <class SH, int DIR>
PTY_DEV void fft_end(const Cta<SH>& c) {
    stage_b<SH, DIR, false>(c);
}
template <class SH, int DIR, class In>
PTY_DEV void fft_2d(const Cta<SH>& c, In& in) {
    fft_begin<SH, DIR>(c, in);
    fft_end<SH, DIR>(c);
}

}  // namespace pty
