// pty_kernels128g2.cuh -- N = 128 forward and adjoint bodies, TWO independent items per CTA.
//
// A CTA of 512 threads is two groups of 256 threads (8 warps, two per SM sub-partition); each group owns
// one (position, mode) item.  The group's 128 x 128 wave lives in tensor memory (256 of the 512 TMEM columns)
// and passes through the registers half at a time: a thread plays two of the four "roles" o = 2 gg + h of the
// 512-thread kernel (pty_fft128.cuh: role = the old thread-group index g), one after the other, 32 complex
// values each.  All layouts (R, K, thread-order workspace arrays) are those of pty_kernels128.cuh with g -> o.
//
//   TMEM, per group: four role blocks of 64 columns; block(q) holds the 32 values role q consumes next.
//     forward exchange : role o writes its fft32 output into block(o) (chunk j = values 8 j .. 8 j + 7 is for
//                        role j); role o' reads chunk o' of every block.
//     inverse exchange : role o' writes the chunk for role q into block(q)[chunk o'] -- exactly the slots it
//                        has just read in the forward direction (a 4 x 4 in-place chunk transpose), so the
//                        k-space pointwise step between a forward and an inverse transform needs no extra space.
//   The two threads of a lane that share a role block are the same lane of warps w and w + 4 of the group:
//   same SM sub-partition, same TMEM lane; their barrier has 64 threads.
//   Shared memory: ONE transpose buffer X (128 x 129 float2) for the CTA, handed back and forth between the
//   groups with named barriers (acquire = bar.sync, release = bar.arrive, 512 = 256 + 256 threads).  Each group
//   holds X for about a third of its time, so the groups settle half a period apart: while one streams its
//   loads, stores and reductions (LSU and latency bound), the other runs butterflies (FP32 pipe bound).
#pragma once
#include "pty_fft128.cuh"
#include "pty_kernels.cuh"

#ifndef PTY_G2_PAIR_NS
#define PTY_G2_PAIR_NS 4   // chunk slots of the pair-sum ring (8 KB each); measured on c4: 2 -> 6.27 ms, 4 -> 6.13 ms, 8 -> 7.30 ms (L1 shrinks)
#endif
#ifndef PTY_G2_D
#define PTY_G2_D 3      // chunks of saved-wave / object rows in flight in the adjoint's streaming step
#endif

namespace pty {

// the memory streams of the adjoint's streaming step, one helper each
PTY_DEV void g2_red_obj(float2* p, float2 v) {
    red_add2(p, v);
}
PTY_DEV float4 g2_ld_psi(const float4* p) {
    return ld_stream4_pinned(p);
}
PTY_DEV float2 g2_ld_obj(const float2* p) {
    return ldg2_pinned(p);
}

PTY_DEV void g2_st_psi(float4* p, float2 a, float2 b) {
    st_stream4(p, a, b);
}

struct G2Smem {
    static constexpr size_t xch_bytes = F128::xch_bytes;
    // twg[128] | per group: Ey, Ex, My, Mx [128 each] float2, red[64] float | TMEM base
    static constexpr size_t group_bytes = 4 * 128 * sizeof(float2) + 64 * sizeof(float);
    // twf[32][12]: FMA-form constants of the forward radix-4 stage (g2_radix4<-1>)
    static constexpr size_t twf_bytes = 32 * 12 * sizeof(float);
    static constexpr size_t bytes = xch_bytes + 128 * sizeof(float2) + 2 * group_bytes + 16 + twf_bytes;
};

struct G2 {
    int tid, t, G, gg, c, smsp;
    float2* X;
    float2* twg;
    const float4* twf;   // [gi][3] float4: (-T1, T1, -T2, T2), (-T3, T3, r31, r31), (g2, g2, g1, g1)
    float2 *Ey, *Ex, *My, *Mx;
    float* red;
    unsigned tl;     // TMEM address: this thread's lane quarter, first column of the group (256 G)
    PTY_DEV unsigned blk(int q) const { return tl + 64u * (unsigned)q; }
    PTY_DEV int kx(int o, int r) const { return 8 * o + (r & 7) + 32 * (r >> 3); }
    PTY_DEV void pair_sync() const {
        tmem_fence_before_sync();
        asm volatile("bar.sync %0, 64;" ::"r"(1 + 4 * G + smsp) : "memory");
        tmem_fence_after_sync();
    }
    PTY_DEV void grp_sync() const { asm volatile("bar.sync %0, 256;" ::"r"(9 + G) : "memory"); }
    PTY_DEV void acquireX() const { asm volatile("bar.sync %0, 512;" ::"r"(11 + G) : "memory"); }
    PTY_DEV void releaseX() const { asm volatile("bar.arrive %0, 512;" ::"r"(11 + (G ^ 1)) : "memory"); }
};

PTY_DEV G2 make_g2(unsigned char* smem) {
    G2 c;
    c.tid = threadIdx.x; c.t = c.tid & 255; c.G = c.tid >> 8; c.gg = (c.tid >> 7) & 1; c.c = c.tid & 127;
    c.smsp = (c.tid >> 5) & 3;
    c.X = reinterpret_cast<float2*>(smem);
    float2* tab = reinterpret_cast<float2*>(smem + G2Smem::xch_bytes);
    c.twg = tab;
    unsigned char* gp = reinterpret_cast<unsigned char*>(tab + 128) + (size_t)c.G * G2Smem::group_bytes;
    float2* gt = reinterpret_cast<float2*>(gp);
    c.Ey = gt; c.Ex = gt + 128; c.My = gt + 256; c.Mx = gt + 384;
    c.red = reinterpret_cast<float*>(gt + 512);
    unsigned* tbase = reinterpret_cast<unsigned*>(reinterpret_cast<unsigned char*>(tab + 128) + 2 * G2Smem::group_bytes);
    if ((threadIdx.x >> 5) == 0) tmem_alloc512(tbase);
    {   // W128^(q gi) = g_q (1 + i T_q), q = 1..3 (forward sign): w u = g (u + T (i u)); a zero cosine (q gi = 32) becomes
        // g = 2^-40, T = -+2^40, which gives -+i u exactly
        float* twf = reinterpret_cast<float*>(tbase + 4);
        c.twf = reinterpret_cast<const float4*>(twf);
        if (c.tid >= 32 && c.tid < 64) fill_twf(c.tid - 32, twf + 12 * (c.tid - 32));
    }
    for (int j = c.tid; j < 128; j += 512) {
        float s, co;
        const int gi = j >> 2, qq = j & 3;
        sincospi_f(2.0f * (float)(qq * gi) / 128.0f, &s, &co);
        c.twg[j] = make_float2(co, -s);
    }
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    c.tl = *tbase + ((32u * (unsigned)c.smsp) << 16) + 256u * (unsigned)c.G;
    return c;
}

PTY_DEV void release_g2(unsigned char* smem) {
    tmem_fence_before_sync();
    __syncthreads();
    float2* tab = reinterpret_cast<float2*>(smem + G2Smem::xch_bytes);
    unsigned* tbase = reinterpret_cast<unsigned*>(reinterpret_cast<unsigned char*>(tab + 128) + 2 * G2Smem::group_bytes);
    if ((threadIdx.x >> 5) == 0) tmem_dealloc512(*tbase);
}

// ------------------------------------------------------------------------------ TMA ring of object rows
// The crop of PAPER.md:75-81 as a TMA gather: the object [Nobj][Nz][H][W] is one 3-D tensor (x, row % 4, row / 4) of
// 8-byte elements, so the rows y = 4 i + o that one role of the FFT needs (layout R) are a box {130, 1, R}: a TMA box
// has to start on a 16-byte boundary of global memory, so it starts at the even column rx & ~1 and is 130 wide (columns
// past the object's edge are zero-filled and never read).  Each
// half-group (128 threads = one role at a time) owns S slots of 4 rows; one elected thread issues the boxes of the
// NEXT role-step (next role, next slice or next item) as soon as the current one has been consumed, so the rows are
// in shared memory long before the multiply needs them -- no registers in flight, no LSU address arithmetic, no L1.
// The remaining rows of a role (32 - 4 S) still come through registers (requested before the preceding transform).
struct G2Ring {
    static constexpr int S = 3, ROWS = 4, COLS = 130;
    static constexpr unsigned slot_bytes = ROWS * COLS * sizeof(float2);            // what one box transfers
    static constexpr unsigned slot_pitch = (slot_bytes + 127) / 128 * 128;          // slots are 128-byte aligned
    static constexpr int slot_elems = slot_pitch / sizeof(float2);
    static constexpr size_t offset = (G2Smem::bytes + 1023) / 1024 * 1024;
    static constexpr size_t bytes = offset + 4 * S * slot_pitch + 4 * 2 * S * sizeof(unsigned long long);
    float2* slots;                        // this half-group's S slots, [S][ROWS][COLS] (pitch slot_elems)
    unsigned long long *full, *empty;     // [S] each
    const CUtensorMap* tm;
    unsigned cpar, ppar;                  // parity of the consumer's next full wait / of the generation the producer fills next
    bool producer;
};

PTY_DEV G2Ring make_g2_ring(unsigned char* smem, const G2& c, const CUtensorMap* tm) {
    G2Ring r;
    const int hg = 2 * c.G + c.gg;        // half-group
    r.slots = reinterpret_cast<float2*>(smem + G2Ring::offset + (size_t)hg * G2Ring::S * G2Ring::slot_pitch);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem + G2Ring::offset + 4 * G2Ring::S * G2Ring::slot_pitch);
    r.full = bars + hg * 2 * G2Ring::S;
    r.empty = r.full + G2Ring::S;
    r.tm = tm;
    r.cpar = 0; r.ppar = 0;
    r.producer = (c.t & 127) == 0;
    if (r.producer) {
#pragma unroll
        for (int k = 0; k < G2Ring::S; ++k) { mbar_init(r.full + k, 1); mbar_init(r.empty + k, 4); }
        mbar_init_fence();
        tma_prefetch_desc(tm);
    }
    __syncthreads();
    return r;
}

// rows (row0 + 4 i), i < 4 S, columns [rx & ~1, +130) -> the half-group's slots (producer thread only)
PTY_DEV void g2_ring_fill(G2Ring& r, int rx, int row0) {
#pragma unroll
    for (int k = 0; k < G2Ring::S; ++k) {
        mbar_wait(r.empty + k, r.ppar ^ 1u);
        mbar_expect_tx(r.full + k, G2Ring::slot_bytes);
        tma_load_3d(r.slots + k * G2Ring::slot_elems, r.tm, rx & ~1, row0 & 3, (row0 >> 2) + G2Ring::ROWS * k, r.full + k);
    }
    r.ppar ^= 1u;
}

// ------------------------------------------------------------------------------ pair sum of the object gradient (a10)
// PTY_FLAG_PAIR_SUM: the two groups of a CTA hold two modes of ONE position, so their contributions conj(psi) g to
// g_object[s, patch] fall on the same pixels.  Group 0 deposits its contribution of every 4-row chunk of the adjoint's
// streaming step in a shared-memory ring, group 1 adds its own and issues the one reduction: half the atomics.  The
// ring (NS chunk slots, full / empty mbarriers, one arrival per warp) is a FIFO over the whole kernel; it bounds how far
// group 0 may run ahead of group 1 (NS chunks), which couples the groups' phases -- the price.
struct G2Pair {
    static constexpr int NS = PTY_G2_PAIR_NS;
    static constexpr int slot_elems = 2 * 4 * 128;                    // [gg][row i][column c] float2
    static constexpr size_t offset = (G2Smem::bytes + 127) / 128 * 128;
    static constexpr size_t bytes = offset + (size_t)NS * slot_elems * sizeof(float2) + 2 * NS * sizeof(unsigned long long);
    float2* slots;
    unsigned long long *full, *empty;
    unsigned q;                                                       // chunks passed so far (same count in both groups)
};
PTY_DEV G2Pair make_g2_pair(unsigned char* smem) {
    G2Pair r;
    r.slots = reinterpret_cast<float2*>(smem + G2Pair::offset);
    r.full = reinterpret_cast<unsigned long long*>(r.slots + G2Pair::NS * G2Pair::slot_elems);
    r.empty = r.full + G2Pair::NS;
    r.q = 0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < G2Pair::NS; ++k) { mbar_init(r.full + k, 8); mbar_init(r.empty + k, 8); }
        mbar_init_fence();
    }
    __syncthreads();
    return r;
}

// crop origin of position b (the same arithmetic as setup_factors: F1 with the clamp of reading R22)
PTY_DEV void g2_crop_origin(const KArgs& A, int b, int& ry, int& rx) {
    const double py = (double)A.positions[2 * b], px = (double)A.positions[2 * b + 1];
    const int iy = (int)floor(py + 0.5), ix = (int)floor(px + 0.5);
    ry = min(max(iy, 0), A.H - 128); rx = min(max(ix, 0), A.W - 128);
}
// first object row of (item, slice 0, role o) in the 3-D view, and its first column
PTY_DEV void g2_item_rows(const KArgs& A, int item, int o, int& row0, int& rx) {
    int b, m, ry;
    size_t obj_off;
    decode_item(A, item, b, m, obj_off);
    g2_crop_origin(A, b, ry, rx);
    row0 = (int)(obj_off / (size_t)A.W) + ry + o;
}

// ------------------------------------------------------------------------------ radix-4 stage with twiddles
// DIR < 0: v[8 q + i] -> twiddle W128^(q (8 o + i)) -> radix-4 over q -> v[8 k2 + i]   (forward)
// DIR > 0: v[8 k2 + i] -> inverse radix-4 over k2 -> conj twiddle -> v[8 q + i]         (inverse)
template <int DIR> PTY_DEV void g2_radix4(const G2& c, int o, float2 (&v)[32]) {
    if constexpr (DIR < 0) {
        // FMA form (pty_fft128.cuh): the three twiddled inputs cost one packed FMA each, their real scales ride on the
        // butterfly's add/sub pairs: 11 packed FMAs per butterfly instead of 12 scalar + 8 packed instructions
        const float4* tf = c.twf + 24 * o;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            bfly4_tw_fma(tf[3 * i], tf[3 * i + 1], tf[3 * i + 2], v[i], v[8 + i], v[16 + i], v[24 + i]);
        }
        return;
    }
    const float4* tw = reinterpret_cast<const float4*>(c.twg + 32 * o);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float4 t01 = tw[2 * i], t23 = tw[2 * i + 1];
        if (DIR < 0) {
            float2 a0 = v[i];
            float2 a1 = cmul_tw(v[8 + i], make_float2(t01.z, t01.w));
            float2 a2 = cmul_tw(v[16 + i], make_float2(t23.x, t23.y));
            float2 a3 = cmul_tw(v[24 + i], make_float2(t23.z, t23.w));
            bfly4<-1>(a0, a1, a2, a3);
            v[i] = a0; v[8 + i] = a1; v[16 + i] = a2; v[24 + i] = a3;
        } else {
            float2 a0 = v[i], a1 = v[8 + i], a2 = v[16 + i], a3 = v[24 + i];
            bfly4<+1>(a0, a1, a2, a3);
            v[i] = a0;
            v[8 + i] = cmulc_tw(make_float2(t01.z, t01.w), a1);
            v[16 + i] = cmulc_tw(make_float2(t23.x, t23.y), a2);
            v[24 + i] = cmulc_tw(make_float2(t23.z, t23.w), a3);
        }
    }
}

// ------------------------------------------------------------------------------ TMEM role blocks
PTY_DEV void g2_ld_own(const G2& c, int o, float2 (&v)[32]) {
#pragma unroll
    for (int j = 0; j < 4; ++j) tmem_ld8(c.blk(o) + 16 * j, v, 8 * j);
    tmem_wait_ld();
}
PTY_DEV void g2_st_own(const G2& c, int o, float2 (&v)[32]) {
#pragma unroll
    for (int j = 0; j < 4; ++j) tmem_st8(c.blk(o) + 16 * j, v, 8 * j);
}
PTY_DEV void g2_ld_slots(const G2& c, int o, float2 (&v)[32]) {
#pragma unroll
    for (int q = 0; q < 4; ++q) tmem_ld8(c.blk(q) + 16 * o, v, 8 * q);
    tmem_wait_ld();
}
PTY_DEV void g2_st_slots(const G2& c, int o, float2 (&v)[32]) {
#pragma unroll
    for (int q = 0; q < 4; ++q) tmem_st8(c.blk(q) + 16 * o, v, 8 * q);
}

// ------------------------------------------------------------------------------ transform phases
// Inverse transform up to the last exchange: role blocks (k space, after the inverse x radix-4) ->
// x fft32^-1 -> X -> y radix-4^-1 -> role blocks.  The caller then runs, per role, g2_ld_own + fft32<+1>.
// FIRST: this is the CTA's very first use of X by group 0 (nothing to acquire).
PTY_DEV void g2_inverse_head(const G2& c, float2 (&v)[32], bool first) {
    constexpr int P = F128::P;
    NoBg bg;
    c.pair_sync();
    if (!first) c.acquireX();
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int o = 2 * c.gg + h;
        g2_ld_own(c, o, v);
        fft32<+1, 0>(v, bg);
        float2* s = c.X + c.c * P + o;
#pragma unroll
        for (int n = 0; n < 32; ++n) s[4 * n] = v[n];
    }
    c.grp_sync();
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int o = 2 * c.gg + h;
        const float2* s = c.X + (8 * o) * P + c.c;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            v[i] = s[i * P];
            v[8 + i] = s[(i + 32) * P];
            v[16 + i] = s[(i + 64) * P];
            v[24 + i] = s[(i + 96) * P];
        }
        if (h == 1) c.releaseX();
        g2_radix4<+1>(c, o, v);
        g2_st_slots(c, o, v);
    }
    tmem_wait_st();
    c.pair_sync();
}

// Forward transform after the per-role fft32<-1> + g2_st_own of the caller: role blocks -> y radix-4 -> X ->
// x fft32 -> role blocks.  The caller then runs, per role, g2_ld_slots + g2_radix4<-1> (k space, layout K).
PTY_DEV void g2_forward_tail(const G2& c, float2 (&v)[32]) {
    constexpr int P = F128::P;
    NoBg bg;
    tmem_wait_st();
    c.pair_sync();
    c.acquireX();
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int o = 2 * c.gg + h;
        g2_ld_slots(c, o, v);
        g2_radix4<-1>(c, o, v);
        float2* s = c.X + (8 * o) * P + c.c;
#pragma unroll
        for (int r = 0; r < 32; ++r) s[((r & 7) + 32 * (r >> 3)) * P] = v[r];
    }
    c.grp_sync();
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int o = 2 * c.gg + h;
        const float2* s = c.X + c.c * P + o;
#pragma unroll
        for (int n2 = 0; n2 < 8; ++n2) {
            v[n2] = s[4 * n2];
            v[8 + n2] = s[4 * (8 + n2)];
            v[16 + n2] = s[4 * (16 + n2)];
            v[24 + n2] = s[4 * (24 + n2)];
        }
        if (h == 1) c.releaseX();
        fft32<-1, 0>(v, bg);
        g2_st_own(c, o, v);
    }
    tmem_wait_st();
    c.pair_sync();
}

PTY_DEV void g2_accumulate(const G2& c, int slot, float v) {
    v = warp_sum(v);
    if (warp_leader()) red_add_shared(c.red + slot, v);
}

// ------------------------------------------------------------------------------ forward (a2-a5)
// item = b MT + n M + m.  The padding item of an odd item count is a GHOST: it runs item n - 1 again with its probe
// (forward) or its seed (adjoint) scaled by 0 and its saved waves in the spare slot `ghost_slot` of the workspace, so
// that every reduction it issues adds zero and no store, reduction or load in these bodies needs a predicate.
// HAT: keep the propagated spectra (tilt / dz gradients); a compile-time switch so that the common no-tilt kernels
// carry neither the code nor the registers of that path.
// TMA: the first 4 S object rows of every role come from the half-group's TMA ring (`ring`; `next_item` = the item this
// group runs after this one, -1 if none: its first rows are requested at the end of this body).
template <bool HAT, bool TMA>
PTY_DEV void fwd_body_g2(const KArgs& A, const G2& c, G2Ring& ring, int item, int slot, float scl, int next_item) {
    constexpr int N = 128, NT = F128::NT;
    int b, m;
    size_t obj_off;
    decode_item(A, item, b, m, obj_off);
    int ry, rx;
    setup_factors<128, 256>(c.t, c.Ey, c.Ex, c.My, c.Mx, c.red, A, b, ry, rx);
    c.grp_sync();
    const size_t NN = (size_t)N * N;
    const size_t bm = (size_t)slot;
    float2 v[32];
    NoBg bg;
    {   // a2 (K): E . P^ -> inverse x radix-4 -> role blocks
        const float2 ey = c.Ey[c.c];
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int o = 2 * c.gg + h;
            const float2* Ph = A.probe_hat + (size_t)m * NN + 128 * o + c.c;
#pragma unroll
            for (int r = 0; r < 32; ++r) v[r] = cmul(cmul(cscale(ldg2(Ph + r * NT), scl), ey), c.Ex[c.kx(o, r)]);
            g2_radix4<+1>(c, o, v);
            g2_st_slots(c, o, v);
        }
        tmem_wait_st();
    }
    bool first = (c.G == 0);
    for (int s = 0; s < A.Nz; ++s) {
        g2_inverse_head(c, v, first);
        first = false;
        // a3 + a4 (R): psi_{s-1} = fft32^-1, keep it, phi_s = O_b[s] psi_{s-1}, first stage of the forward y transform
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int o = 2 * c.gg + (TMA ? h : (h ^ c.G));   // group 1 takes its roles in the opposite order: its object rows are then the ones group 0 read last (L1 hits)
            const float2* obj = A.object + obj_off + ((size_t)s * A.H + ry + o) * A.W + rx + c.c;
            const size_t ostride = (size_t)4 * A.W;
            float2 oa[8], ob[8];
            float4* save = reinterpret_cast<float4*>(A.ws_psi + (bm * A.Nz + s) * NN) + 128 * o + c.c;
#define PTY_G2_SAVE(J)                                                                                  \
            { _Pragma("unroll") for (int i = 0; i < 8; i += 2)                                          \
                g2_st_psi(save + (4 * J + i / 2) * NT, v[8 * J + i], v[8 * J + i + 1]); }
            if constexpr (TMA) {
                // rows 0..11 from the ring, 12..19 (oa) and 20..27 (ob) requested now, 28..31 once oa[0..3] are free
                static_assert(G2Ring::S == 3 && G2Ring::ROWS == 4, "row split of the TMA path");
#pragma unroll
                for (int i = 0; i < 8; ++i) oa[i] = g2_ld_obj(obj + (size_t)(12 + i) * ostride);
#pragma unroll
                for (int i = 0; i < 8; ++i) ob[i] = g2_ld_obj(obj + (size_t)(20 + i) * ostride);
                g2_ld_own(c, o, v);
                fft32<+1, 0>(v, bg);
                const float2* rs = ring.slots + (rx & 1) + c.c;
                constexpr int RS = G2Ring::slot_elems, RC = G2Ring::COLS;
                PTY_G2_SAVE(0)
                mbar_wait(ring.full + 0, ring.cpar);
#pragma unroll
                for (int i = 0; i < 4; ++i) v[i] = cmul(v[i], rs[i * RC]);
                mbar_wait(ring.full + 1, ring.cpar);
#pragma unroll
                for (int i = 0; i < 4; ++i) v[4 + i] = cmul(v[4 + i], rs[RS + i * RC]);
                PTY_G2_SAVE(1)
                mbar_wait(ring.full + 2, ring.cpar);
#pragma unroll
                for (int i = 0; i < 4; ++i) v[8 + i] = cmul(v[8 + i], rs[2 * RS + i * RC]);
                ring.cpar ^= 1u;
                __syncwarp();
                if (warp_leader()) { mbar_arrive(ring.empty + 0); mbar_arrive(ring.empty + 1); mbar_arrive(ring.empty + 2); }
#pragma unroll
                for (int i = 0; i < 4; ++i) v[12 + i] = cmul(v[12 + i], oa[i]);
#pragma unroll
                for (int i = 0; i < 4; ++i) oa[i] = g2_ld_obj(obj + (size_t)(28 + i) * ostride);
                PTY_G2_SAVE(2)
#pragma unroll
                for (int i = 0; i < 4; ++i) v[16 + i] = cmul(v[16 + i], oa[4 + i]);
#pragma unroll
                for (int i = 0; i < 4; ++i) v[20 + i] = cmul(v[20 + i], ob[i]);
                PTY_G2_SAVE(3)
#pragma unroll
                for (int i = 0; i < 4; ++i) v[24 + i] = cmul(v[24 + i], ob[4 + i]);
#pragma unroll
                for (int i = 0; i < 4; ++i) v[28 + i] = cmul(v[28 + i], oa[i]);
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) oa[i] = g2_ld_obj(obj + (size_t)i * ostride);
                g2_ld_own(c, o, v);
                fft32<+1, 0>(v, bg);
#define PTY_G2_CHUNK(J, CUR, NXT)                                                                       \
                {                                                                                       \
                    if (J < 3) { _Pragma("unroll") for (int i = 0; i < 8; ++i)                          \
                        NXT[i] = g2_ld_obj(obj + (size_t)(8 * (J + 1) + i) * ostride); }                \
                    PTY_G2_SAVE(J)                                                                      \
                    _Pragma("unroll") for (int i = 0; i < 8; ++i) v[8 * J + i] = cmul(v[8 * J + i], CUR[i]); \
                }
                PTY_G2_CHUNK(0, oa, ob) PTY_G2_CHUNK(1, ob, oa) PTY_G2_CHUNK(2, oa, ob) PTY_G2_CHUNK(3, ob, oa)
#undef PTY_G2_CHUNK
            }
#undef PTY_G2_SAVE
            fft32<-1, 0>(v, bg);
            g2_st_own(c, o, v);
            if constexpr (TMA) {
                // the ring's slots are free again (every warp of the half-group has arrived or will shortly): request the
                // rows of the next role-step -- the other role of this slice, the first role of the next slice, or of the
                // next item
                if (ring.producer) {
                    const int row_now = (int)(obj_off / (size_t)A.W) + s * A.H + ry + o;
                    if (h == 0) g2_ring_fill(ring, rx, row_now + 1);
                    else if (s + 1 < A.Nz) g2_ring_fill(ring, rx, row_now - 1 + A.H);
                    else if (next_item >= 0) {
                        int row0, rxn;
                        g2_item_rows(A, next_item, 2 * c.gg, row0, rxn);
                        g2_ring_fill(ring, rxn, row0);
                    }
                }
            }
        }
        g2_forward_tail(c, v);
        if (s == A.Nz - 1) break;
        // a4 (K): propagator, inverse x radix-4, in-place slots
        const float2 my = c.My[c.c];
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int o = 2 * c.gg + h;
            g2_ld_slots(c, o, v);
            g2_radix4<-1>(c, o, v);
            float2* hat = HAT ? A.ws_hat + (bm * (A.Nz - 1) + s) * NN + 128 * o + c.c : nullptr;
#pragma unroll
            for (int r = 0; r < 32; ++r) {
                v[r] = cmul(v[r], cmul(my, c.Mx[c.kx(o, r)]));
                if (HAT) st_stream2(hat + r * NT, v[r]);
            }
            g2_radix4<+1>(c, o, v);
            g2_st_slots(c, o, v);
        }
        tmem_wait_st();
    }
    // a5 (K): Psi = F[phi_Nz] / N, I += |Psi|^2.  I is kept in thread order as pairs, [r / 2][128 o + ky][r & 1]
    // (layout K: register r of role o holds k_x = 8 o + (r & 7) + 32 (r >> 3)): one 8-byte vector RED per two
    // registers, lane-contiguous, no transpose; pty_loss_seed128_kernel<true> reads it in that order.
    float2* Ib = reinterpret_cast<float2*>(A.I + (size_t)b * NN);
#pragma unroll 1
    for (int h = 0; h < 2; ++h) {
        const int o = 2 * c.gg + h;
        g2_ld_slots(c, o, v);
        g2_radix4<-1>(c, o, v);
        float2* Psi = A.ws_Psi + bm * NN + 128 * o + c.c;
#pragma unroll
        for (int r = 0; r < 32; r += 2) {
            const float2 p0 = cscale(v[r], 1.0f / N), p1 = cscale(v[r + 1], 1.0f / N);
            st_stream2(Psi + r * NT, p0);
            st_stream2(Psi + (r + 1) * NT, p1);
            red_add2(Ib + (r >> 1) * NT + 128 * o + c.c, make_float2(p0.x * p0.x + p0.y * p0.y, p1.x * p1.x + p1.y * p1.y));
        }
    }
    if (c.G == 0) c.acquireX();      // consume group 1's last release
}

// ------------------------------------------------------------------------------ adjoint (a7-a13)
template <bool HAT, bool PAIR> PTY_DEV void bwd_body_g2(const KArgs& A, const G2& c, G2Pair& pr, int item, int slot, float scl) {
    constexpr int N = 128, NT = F128::NT;
    int b, m;
    size_t obj_off;
    decode_item(A, item, b, m, obj_off);
    int ry, rx;
    setup_factors<128, 256>(c.t, c.Ey, c.Ex, c.My, c.Mx, c.red, A, b, ry, rx);
    c.grp_sync();
    const size_t NN = (size_t)N * N;
    const size_t bm = (size_t)slot;
    float2 v[32];
    NoBg bg;
    {   // a7, a8 (K): g_Psi = w Psi, inverse x radix-4 -> role blocks
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int o = 2 * c.gg + h;
            const float2* Psi = A.ws_Psi + bm * NN + 128 * o + c.c;
            const float* Wt = A.seed_w + (size_t)b * NN + 128 * o + c.c;
#pragma unroll
            for (int r = 0; r < 32; ++r) v[r] = cscale(ld_stream2(Psi + r * NT), ldg1(Wt + r * NT) * scl);
            g2_radix4<+1>(c, o, v);
            g2_st_slots(c, o, v);
        }
        tmem_wait_st();
    }
    float acc_ky = 0.f, acc_kx = 0.f, acc_k2 = 0.f;
    bool first = (c.G == 0);
    for (int s = A.Nz - 1; s >= 0; --s) {
        g2_inverse_head(c, v, first);
        first = false;
        // a9, a10 (R): g = fft32^-1; g_object patch += conj(psi_{s-1}) g; g <- conj(O_b[s]) g; forward y first stage.
        // Park-then-stream: both roles' g goes back to its TMEM block first, which frees the 64 wave registers;
        // the pointwise step then streams over the 16 chunks of 4 rows (two roles x 8) with the saved wave (HBM
        // stream) and the object rows D chunks ahead in registers and g one chunk ahead from TMEM.  (Requesting the first
        // D saved-wave chunks before the park phase's inverse fft32 measured -4 %: round 2.)
        constexpr int D = PTY_G2_D;
        const float4* psi0 = reinterpret_cast<const float4*>(A.ws_psi + (bm * A.Nz + s) * NN) + 256 * c.gg + c.c;
        float4 pb[D][2];
        // group 1 streams its two roles in the opposite order: the object rows it reads are then the ones group 0 (same
        // position, the neighbouring mode) has read last, and they are still in L1
        const int fl = !PAIR ? c.G : 0;     // pair sum: both groups must walk the rows in one order
        const int pr0 = fl ? 128 : 0, pr1 = 128 - pr0;                      // saved-wave offset of the first / second role
        const size_t or0 = fl ? (size_t)A.W : 0, or1 = (size_t)A.W - or0;   // object-row offset
        const unsigned tr0 = fl ? 64u : 0u, tr1 = 64u - tr0;                // TMEM role block
#define PTY_G2_ISSUE_PSI(J)                                                                               \
        {                                                                                                 \
            const float4* pp_ = psi0 + ((J) >> 3 ? pr1 : pr0) + (size_t)(2 * ((J) & 7)) * NT;             \
            pb[(J) % D][0] = g2_ld_psi(pp_);                                                              \
            pb[(J) % D][1] = g2_ld_psi(pp_ + NT);                                                         \
        }
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int o = 2 * c.gg + h;
            g2_ld_own(c, o, v);
            fft32<+1, 0>(v, bg);
            g2_st_own(c, o, v);
        }
        tmem_wait_st();
        {
            const size_t ostride = (size_t)4 * A.W;
            const float2* obj0 = A.object + obj_off + ((size_t)s * A.H + ry + 2 * c.gg) * A.W + rx + c.c;
            float2* gobj0 = A.g_object + obj_off + ((size_t)s * A.H + ry + 2 * c.gg) * A.W + rx + c.c;
            const unsigned tb0 = c.blk(2 * c.gg);
            float2 ob[D][4];
            float2 gb[2][4];
#define PTY_G2_ISSUE_OBJ(J)                                                                               \
            {                                                                                             \
                const float2* oo_ = obj0 + ((J) >> 3 ? or1 : or0) + (size_t)(4 * ((J) & 7)) * ostride;    \
                _Pragma("unroll") for (int i = 0; i < 4; ++i) ob[(J) % D][i] = g2_ld_obj(oo_ + (size_t)i * ostride); \
            }
#define PTY_G2_ISSUE(J) { PTY_G2_ISSUE_PSI(J) PTY_G2_ISSUE_OBJ(J) }   // one statement: used under `if (D > n)`
#define PTY_G2_STEP(J)                                                                                    \
            {                                                                                             \
                tmem_wait_ld();                                                                           \
                if ((J) < 15) tmem_ld4(tb0 + (((J) + 1) >> 3 ? tr1 : tr0) + 8u * (((J) + 1) & 7), gb[((J) + 1) & 1]); \
                float2* go_ = gobj0 + ((J) >> 3 ? or1 : or0) + (size_t)(4 * ((J) & 7)) * ostride;         \
                float2 ct_[4];                                                                            \
                _Pragma("unroll") for (int i = 0; i < 4; ++i) {                                           \
                    const float4 q_ = pb[(J) % D][i >> 1];                                                \
                    const float2 ps = (i & 1) ? make_float2(q_.z, q_.w) : make_float2(q_.x, q_.y);        \
                    const float2 g_ = gb[(J) & 1][i];                                                     \
                    ct_[i] = cmulc(ps, g_);                                                               \
                    gb[(J) & 1][i] = cmulc(ob[(J) % D][i], g_);                                           \
                }                                                                                         \
                if constexpr (PAIR) {                                                                     \
                    const unsigned k_ = pr.q % G2Pair::NS, ph_ = (pr.q / G2Pair::NS) & 1u;                \
                    float2* sl_ = pr.slots + k_ * G2Pair::slot_elems + 512 * c.gg + c.c;                  \
                    if (c.G == 0) {                                                                       \
                        mbar_wait(pr.empty + k_, ph_ ^ 1u);                                               \
                        _Pragma("unroll") for (int i = 0; i < 4; ++i) sl_[128 * i] = ct_[i];              \
                        __syncwarp();                                                                     \
                        if (warp_leader()) mbar_arrive(pr.full + k_);                                     \
                    } else {                                                                              \
                        mbar_wait(pr.full + k_, ph_);                                                     \
                        _Pragma("unroll") for (int i = 0; i < 4; ++i)                                     \
                            g2_red_obj(go_ + (size_t)i * ostride, cadd(ct_[i], sl_[128 * i]));            \
                        __syncwarp();                                                                     \
                        if (warp_leader()) mbar_arrive(pr.empty + k_);                                    \
                    }                                                                                     \
                    ++pr.q;                                                                               \
                } else {                                                                                  \
                    _Pragma("unroll") for (int i = 0; i < 4; ++i) g2_red_obj(go_ + (size_t)i * ostride, ct_[i]); \
                }                                                                                         \
                tmem_st4(tb0 + ((J) >> 3 ? tr1 : tr0) + 8u * ((J) & 7), gb[(J) & 1]);                     \
                if ((J) + D < 16) { PTY_G2_ISSUE_PSI((J) + D) PTY_G2_ISSUE_OBJ((J) + D) }                 \
            }
            PTY_G2_ISSUE(0) PTY_G2_ISSUE(1) PTY_G2_ISSUE(2)
            if (D > 3) PTY_G2_ISSUE(3)
            if (D > 4) PTY_G2_ISSUE(4)
            if (D > 5) PTY_G2_ISSUE(5)
            tmem_ld4(tb0 + tr0, gb[0]);
            PTY_G2_STEP(0) PTY_G2_STEP(1) PTY_G2_STEP(2) PTY_G2_STEP(3) PTY_G2_STEP(4) PTY_G2_STEP(5)
            PTY_G2_STEP(6) PTY_G2_STEP(7) PTY_G2_STEP(8) PTY_G2_STEP(9) PTY_G2_STEP(10) PTY_G2_STEP(11)
            PTY_G2_STEP(12) PTY_G2_STEP(13) PTY_G2_STEP(14) PTY_G2_STEP(15)
#undef PTY_G2_STEP
#undef PTY_G2_ISSUE
#undef PTY_G2_ISSUE_OBJ
#undef PTY_G2_ISSUE_PSI
        }
        tmem_wait_st();
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int o = 2 * c.gg + h;
            g2_ld_own(c, o, v);
            fft32<-1, 0>(v, bg);
            g2_st_own(c, o, v);
        }
        g2_forward_tail(c, v);
        if (s == 0) break;
        // a9, a13 (K): D-sums against the kept spectrum, conj(M), inverse x radix-4, in-place slots
        const float2 my = c.My[c.c];
        const float kyf = kp_of<N>(c.c);
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int o = 2 * c.gg + h;
            g2_ld_slots(c, o, v);
            g2_radix4<-1>(c, o, v);
            if (HAT) {
                const float2* hat = A.ws_hat + (bm * (A.Nz - 1) + (s - 1)) * NN + 128 * o + c.c;
#pragma unroll
                for (int r = 0; r < 32; ++r) {
                    const float2 hs = ld_stream2(hat + r * NT);
                    const float d = hs.x * v[r].y - hs.y * v[r].x;          // Im(conj(psi^) g^)
                    const float kxf = kp_of<N>(c.kx(o, r));
                    acc_ky += d * kyf;
                    acc_kx += d * kxf;
                    acc_k2 += d * (kyf * kyf + kxf * kxf);
                }
            }
#pragma unroll
            for (int r = 0; r < 32; ++r) v[r] = cmulc(cmul(my, c.Mx[c.kx(o, r)]), v[r]);
            g2_radix4<+1>(c, o, v);
            g2_st_slots(c, o, v);
        }
        tmem_wait_st();
    }
    // a11, a12 (K): g^_0 = F[g_psi0]; probe-gradient accumulation and the position gradient
    float accy = 0.f, accx = 0.f;
    {
        const float2 ey = c.Ey[c.c];
        const float kyf = kp_of<N>(c.c);
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            const int o = 2 * c.gg + h;
            g2_ld_slots(c, o, v);
            g2_radix4<-1>(c, o, v);
            const float2* Ph = A.probe_hat + (size_t)m * NN + 128 * o + c.c;
            float2* GP = A.GP_hat + (size_t)m * NN + 128 * o + c.c;
#pragma unroll
            for (int r = 0; r < 32; ++r) {
                const int kx = c.kx(o, r);
                const float2 gg = v[r];
                const float2 e = cmul(ey, c.Ex[kx]);                     // E / N
                red_add2(GP + r * NT, cmulc(e, gg));
                const float2 ep = cmul(e, ldg2(Ph + r * NT));
                const float t = gg.x * ep.y - gg.y * ep.x;               // Im(conj(g^_0) E P^)
                accy += kyf * t;
                accx += kp_of<N>(kx) * t;
            }
        }
    }
    g2_accumulate(c, 0, accy);
    g2_accumulate(c, 1, accx);
    if (HAT) {
        g2_accumulate(c, 2, acc_ky);
        g2_accumulate(c, 3, acc_kx);
        g2_accumulate(c, 4, acc_k2);
    }
    c.grp_sync();
    if (c.t == 0) {
        const float two_pi = 6.283185307179586f;
        if (A.g_pos) {
            red_add(A.g_pos + 2 * b, two_pi * c.red[0]);
            red_add(A.g_pos + 2 * b + 1, two_pi * c.red[1]);
        }
        if (HAT) {
            red_add(A.dsum + 4 * b, c.red[2]);
            red_add(A.dsum + 4 * b + 1, c.red[3]);
            red_add(A.dsum + 4 * b + 2, c.red[4]);
        }
    }
    if (c.G == 0) c.acquireX();      // consume group 1's last release
}

}  // namespace pty
