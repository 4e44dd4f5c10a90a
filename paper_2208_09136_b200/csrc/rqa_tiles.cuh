// rqa_tiles.cuh — what the two full passes over the upper triangle share (the counting pass of rqa_eps_for_rr
// in rqa_select.cu and the diagonal scan of rqa_line_hist in rqa_line.cu): the tiling of the triangle, the
// staging of the two series windows in shared memory, the sliding-window cell distance and the bucket function
// of the level tables.  Internal to librqa.so; nothing here is shared with the oracle.
//
// Tiling.  The recurrence plot's upper triangle (only j > i is visited, R_ij is computed on the
// fly) is cut into diagonal blocks of LW = 512 adjacent diagonals o = j - i (one per thread), and every diagonal
// block into chunks of L consecutive positions i.  A tile = (diagonal block, chunk).  The lanes of a warp sit on
// 32 adjacent diagonals at the same position i, so y[i] is a shared-memory broadcast and y[i + o] is 32
// consecutive words: no bank conflicts.
//
// Distance.  With the delay view x_i[c] = y[i + c*tau] the max-norm distance along a diagonal is a
// sliding maximum over e_i = |y_i - y_{i+o}|, and the squared Euclidean distance a sliding sum in the
// fixed order c = 0..m-1 (reading S13): one new element per cell, kept in a register ring.
#pragma once

#include <utility>

#include "rqa_common.cuh"

namespace rqa {

constexpr int LW = 512;          // diagonals per tile = threads per block
constexpr int NB = 4096;         // buckets of a level look-up table
constexpr int GK = 32;           // thresholds (or brackets) per group = per full pass
constexpr int MAX_SPAN = 4096;   // largest (m-1)*tau the tiled kernels stage in shared memory
constexpr unsigned FULL = 0xffffffffu;

// bucket(d) = bits(fmaf(min(d, dcap), scale, 2^23)) - bits(2^23): adding 2^23 leaves round(d * scale) in the low
// mantissa bits, i.e. an exactly rounded, monotone map of [0, dcap] onto the integers 0..nb-1 in one FMA, for
// thresholds of any magnitude (scale = (nb - 1.5) / dcap is an ordinary float).  The subtraction folds into the table's
// base address.
constexpr uint32_t BUCKET_MAGIC_BITS = 0x4B000000u;              // bits of 8388608.0f = 2^23
__device__ __forceinline__ uint32_t bucket_bits(float d, float dcap, float scale) {      // bucket + BUCKET_MAGIC_BITS
    return __float_as_uint(__fmaf_rn(fminf(d, dcap), scale, 8388608.0f));
}
__device__ __forceinline__ uint32_t bucket_of(float d, float dcap, float scale) {
    return bucket_bits(d, dcap, scale) - BUCKET_MAGIC_BITS;
}

// Largest scale for which bucket_of(dcap) <= nb-1 (nb <= 2^22).  Denormal-small dcap: the scale saturates, every
// distance falls into the lowest buckets and the tables' refinement loops do the work.
__device__ inline float bucket_scale(float dcap, int nb = NB) {
    double sc = ((double)nb - 1.5) / (double)dcap;
    float scale = sc > 3.0e38 ? 3.0e38f : (float)sc;
    while (scale > 0.0f && bucket_of(dcap, dcap, scale) > (uint32_t)(nb - 1)) scale = nextafterf(scale, 0.0f);
    return scale;
}

// Tiling of the triangle of nd = N' - w + 1 "points" (diagonals w..N'-1) for one part of a (possibly split) call.
// Diagonal block ob holds LW adjacent diagonals; part `part` of `parts` owns the blocks ob = part, part + parts, ...
// (interleaved: every part gets long and short diagonals).  Local block q <-> ob = part + q*parts.  A tile is T
// consecutive positions of one diagonal block.
struct Tiling {
    int64_t nd;       // points of the counted triangle
    int64_t T;        // cells per tile along the diagonals
    int part, parts;
    int n_ob;         // diagonal blocks of the whole triangle
    int n_obl;        // ... owned by this part
    uint64_t tiles;   // tiles of this part (one series)
};
inline Tiling make_tiling(int64_t nd, int64_t T, int part, int parts) {
    Tiling t{};
    t.nd = nd; t.T = T; t.part = part; t.parts = parts;
    t.n_ob = (int)((nd - 1 + LW - 1) / LW);
    t.n_obl = t.n_ob > part ? (t.n_ob - part + parts - 1) / parts : 0;
    t.tiles = 0;
    for (int q = 0; q < t.n_obl; ++q) t.tiles += (uint64_t)((nd - 1 - (int64_t)LW * (part + (int64_t)q * parts) + T - 1) / T);
    return t;
}
// tile_start[q] = number of tiles in the local diagonal blocks before q (q = 0..n_obl), computed on the device.
rqa_status launch_tile_table(const Tiling& t, uint32_t* tile_start, cudaStream_t s);

#ifdef __CUDACC__
// Shared-memory accesses of the tiled passes' inner loops go through 32-bit shared-window addresses and explicit .shared
// instructions: with generic pointers the compiler re-derives the window base inside the loop when registers are tight.
// pin(): an identity shuffle (call it with the whole warp converged).  ptxas lowers a shared symbol's address to
// S2R SR_CgaCtaId + LEA and, being "cheap", rematerialises that per use inside the loop; a shuffle result is kept.
__device__ __forceinline__ uint32_t pin(uint32_t x) { return __shfl_sync(0xffffffffu, x, threadIdx.x & 31); }
__device__ __forceinline__ unsigned long long pin64(unsigned long long x) { return __shfl_sync(0xffffffffu, x, threadIdx.x & 31); }
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return pin((uint32_t)__cvta_generic_to_shared(p)); }
__device__ __forceinline__ float lds_f32(uint32_t a) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }
__device__ __forceinline__ void lds_f32_u32(uint32_t a, float& x, uint32_t& y) { asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=f"(x), "=r"(y) : "r"(a)); }
__device__ __forceinline__ void lds_v4f(uint32_t a, float& x, float& y, float& z, float& w) { asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x), "=f"(y), "=f"(z), "=f"(w) : "r"(a)); }
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ uint32_t lds_u16(uint32_t a) { uint32_t v; asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ uint32_t lds_u8(uint32_t a) { uint32_t v; asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ void sts_u32(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" :: "r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts_u16(uint32_t a, uint32_t v) { asm volatile("st.shared.u16 [%0], %1;" :: "r"(a), "h"((unsigned short)v) : "memory"); }
__device__ __forceinline__ void sts_v4(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) { asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" :: "r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory"); }
__device__ __forceinline__ uint32_t atom_u32(uint32_t a, uint32_t v) { uint32_t o; asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(o) : "r"(a), "r"(v) : "memory"); return o; }
__device__ __forceinline__ void red_u32(uint32_t a, uint32_t v) { asm volatile("red.shared.add.u32 [%0], %1;" :: "r"(a), "r"(v) : "memory"); }

// ---- bulk asynchronous copies global -> shared (the TMA engine's 1-D path) completing on an mbarrier
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" :: "r"(bar), "r"(parity) : "memory");
}
// dst (shared, 16-byte aligned), src (global, 16-byte aligned), bytes a multiple of 16
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// orders earlier generic-proxy accesses of shared memory before later async-proxy (bulk copy) writes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Which diagonal block does `tile` belong to?  (block-wide search; the caller syncs before reading *s_ob)
__device__ __forceinline__ void find_diagonal_block(const uint32_t* __restrict__ tile_start, int n_ob, uint32_t tile,
                                                    int* s_ob) {
    for (int q = threadIdx.x; q < n_ob; q += LW)
        if (tile_start[q] <= tile && tile < tile_start[q + 1]) *s_ob = q;
}

// Window lengths (floats) for a chunk of L positions, embedding span (m-1)*tau and W warm-up cells before the chunk:
// i-side window y[s-W .. s-W+LA), j-side window y[s-W+o0 .. s-W+o0+LB).
// ps = point stride in floats (1 for a delay view, m for materialised row-major points); span = (m-1) * coord stride.
// WSLACK: the last super-step of a chunk starts before cell L and touches up to U - 1 cells plus S - 1 ring elements
// beyond it (U <= 12 cells per super-step, S - 1 <= span), loaded before the guards look at them.
constexpr int WSLACK = 16;
__host__ __device__ inline int window_la(int L, int span, int W, int ps = 1) { return ((L + W + WSLACK) * ps + 2 * span + 3) & ~3; }
__host__ __device__ inline int window_lb(int L, int span, int W, int ps = 1) { return ((L + W + WSLACK + LW) * ps + 2 * span + 3) & ~3; }

// Stage the two windows of series `y` (ny samples); samples outside the series read as 0 (their cells are never
// counted).
__device__ __forceinline__ void stage_windows(const float* __restrict__ y, int64_t ny, int64_t start_a, int64_t start_b,
                                              float* ya_s, int LA, float* yb_s, int LB) {
    for (int x = threadIdx.x; x < LA; x += LW) {
        int64_t gi = start_a + x;
        ya_s[x] = (gi >= 0 && gi < ny) ? y[gi] : 0.0f;
    }
    for (int x = threadIdx.x; x < LB; x += LW) {
        int64_t gi = start_b + x;
        yb_s[x] = (gi >= 0 && gi < ny) ? y[gi] : 0.0f;
    }
}

// Cell distances along one diagonal from the staged windows.  W = warm-up cells before the chunk (cell t of the
// chunk reads window index t + W).  M > 0: compile-time (M, TAU), sliding window over a register ring of
// S = (M-1)*TAU + 1 elements.  M == 0: run-time (m, tau), recomputed from the windows for every cell.
// The two window addresses are CURSORS: they point at the element of the first cell of the current super-step
// (seek / advance), so that every access inside a super-step is cursor + a compile-time offset.
// VEC (register-ring variants only): the i-side window is read four elements per load (all lanes read the same
// address: one broadcast wavefront instead of four).  The caller places the window so that the element pushed by the first
// cell of a super-step (cursor + S - 1) is 16-byte aligned, and uses super-steps of a multiple of 4 cells.
template <int NORM, int M, int TAU, int W, bool VEC = false>
struct CellDist {
    static constexpr int S = M > 0 ? (M - 1) * TAU + 1 : 1;
    static_assert(!VEC || M > 0, "vector loads belong to the register-ring variants");
    float ring[S];
    float ya4[VEC ? 4 : 1];     // VEC: the four i-side elements of the current group of cells
    uint32_t ya;                // shared-window address of the i-side window element of cell t0
    uint32_t yb;                // ... of the j-side window, already offset by the thread's diagonal
    int m, tau;                 // M == 0: run-time dimension and coordinate stride (floats)
    int ps;                     // M == 0: point stride (floats); the register-ring variants are delay views, stride 1

    __device__ __forceinline__ int pstride() const { return M > 0 ? 1 : ps; }
    // ya_org, yb_org: addresses of window index 0 (cell -W); afterwards the cursors stand at cell t0
    __device__ __forceinline__ void seek(uint32_t ya_org, uint32_t yb_org, int t0) {
        ya = ya_org + 4 * (t0 + W) * pstride();
        yb = yb_org + 4 * (t0 + W) * pstride();
    }
    __device__ __forceinline__ void advance(int cells) { ya += 4 * cells * pstride(); yb += 4 * cells * pstride(); }

    // element x cells after the cursor
    __device__ __forceinline__ float elem(int x) const {
        // max norm: the signed difference is kept, |.| is an operand modifier of the maximum in distance()
        float diff = __fsub_rn(lds_f32(ya + 4 * x), lds_f32(yb + 4 * x));
        return NORM == RQA_NORM_MAX ? diff : __fmul_rn(diff, diff);
    }
    // Before the first cell (cursor on it; it must be processed at ring phase R = 0) the ring holds e_t .. e_{t+S-2}.
    __device__ __forceinline__ void prime() {
#pragma unroll
        for (int x = 0; x < (M > 0 ? S - 1 : 0); ++x) ring[x] = elem(x);
    }
    // R = offset of the cell from the cursor = its ring phase (static); pushes e_{t+S-1}
    template <int R>
    __device__ __forceinline__ void push() {
        if (M > 0 && VEC) {
            if (R % 4 == 0) lds_v4f(ya + 4 * (R + S - 1), ya4[0], ya4[1], ya4[2], ya4[3]);
            float diff = __fsub_rn(ya4[R % 4], lds_f32(yb + 4 * (R + S - 1)));
            ring[(R + S - 1) % S] = NORM == RQA_NORM_MAX ? diff : __fmul_rn(diff, diff);
        } else if (M > 0) {
            ring[(R + S - 1) % S] = elem(R + S - 1);
        }
    }
    template <int R>
    __device__ __forceinline__ float distance() const {
        if (M == 0) {
            float d = elem(R * ps);
            if (NORM == RQA_NORM_MAX) d = fabsf(d);
            for (int c = 1; c < m; ++c) {
                float x = elem(R * ps + c * tau);
                d = NORM == RQA_NORM_MAX ? fmaxf(d, fabsf(x)) : __fadd_rn(d, x);
            }
            return NORM == RQA_NORM_MAX ? d : __fsqrt_rn(d);
        }
        float d = ring[R % S];
        if (NORM == RQA_NORM_MAX) d = fabsf(d);
#pragma unroll
        for (int c = 1; c < M; ++c) {
            float x = ring[(R + c * TAU) % S];
            d = NORM == RQA_NORM_MAX ? fmaxf(d, fabsf(x)) : __fadd_rn(d, x);
        }
        return NORM == RQA_NORM_MAX ? d : __fsqrt_rn(d);
    }
};
#endif

}  // namespace rqa
