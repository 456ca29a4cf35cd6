// bg_tables.cuh -- compile-time work lists for the tiled Berends-Giele kernel (bg_tile.cuh).
//
// The sums over splittings of Eq.(6) are flattened, level by level, into a
// list of ITEMS: for the current (i..j) of length L, in la-major order, the 3-gluon split
// (i..k | k+1..j), k = i+la-1, followed by the 4-gluon splits (i..k | k+1..l | l+1..j),
// l = k+lb.  The list of a level is cut into W contiguous chunks of (nearly) equal weight,
// one per warp of the tile, so the warps of a block stay balanced whatever the number of
// currents at that level.  A chunk boundary may fall inside a current; such a current gets
// its partial sums combined by a "gather job" after a block barrier.
//
// Everything here is evaluated by the compiler (constexpr) and lands in constant memory:
// the kernel reads it with warp-uniform indices, and its code is a short loop over items
// instead of an unrolled body per splitting (the unrolled form of round 1 was bound by
// instruction fetch: profiles/r01a_cfg2_sweep_w4_metrics.txt, gcc instruction requests 98 %).
#pragma once
#include <stdint.h>

namespace bg {

// flags of an item (bits 24..31 of word x)
constexpr uint32_t IT_KIND4 = 1u;       // 0: 3-gluon split, 1: 4-gluon split
constexpr uint32_t IT_LOAD_A = 2u;      // left factor J(i..k) differs from the previous item's
constexpr uint32_t IT_SEG_START = 4u;   // first item of a (current, chunk) segment
constexpr uint32_t IT_SEG_END = 8u;     // last item of a segment
constexpr uint32_t IT_COMPLETE = 16u;   // at SEG_END: the segment is the whole current -> finish inline
constexpr uint32_t IT_TOP = 32u;        // the current is J(1..n-1): no propagator, amplitude

constexpr int kWeight3 = 8, kWeight4 = 3, kWeightFinish = 10;

struct TileItem {
    // x: a_row | b_row << 8 | c << 16 | flags << 24
    //      3-split: a = J(i..k), b = J(k+1..j), c = k (index of the doubled prefix sum PS2_k)
    //      4-split: a = J(i..k), b = J(k+1..l) (the middle factor), c = row of J(l+1..j)
    // y: lo | hi << 8 | own_row << 16 | slot << 24
    //      lo = i-1, hi = j: P_{i,j} = PS_hi - PS_lo;  own_row: where J(i..j) is stored;
    //      slot: scratch slot of a partial segment
    uint32_t x, y;
};

// The form the kernel reads: byte offsets into the per-point vector record, ready for use as
// [base + offset] operands (independent of W), and the chunk-dependent flags on the side.
struct alignas(16) TileOff {
    uint32_t a, b, c;      // byte offsets of the three vector rows (c: PS2_k row for a 3-split)
    uint32_t uv;           // 3-split: byte offset of U_A | byte offset of V_B << 16 in the lane's scalar column
};

template <int N, int W>
struct TileTables {
    static constexpr int M = N - 1;
    static constexpr int NITEMS = N * (N - 1) * (N - 2) / 6 + N * (N - 1) * (N - 2) * (N - 3) / 24;
    static constexpr int MAXJOBS = W;
    TileItem items[NITEMS];
    uint16_t beg[M + 1][W + 1];          // warp w of level L owns items [beg[L][w], beg[L][w+1])
    TileItem jobs[M + 1][MAXJOBS];       // x: slot mask;  y: as in TileItem (slot unused)
    uint8_t njobs[M + 1];
};

// what lands in constant memory
template <int N, int W>
struct TileProgram {
    static constexpr int M = N - 1;
    static constexpr int NITEMS = TileTables<N, W>::NITEMS;
    TileOff off[NITEMS];
    uint32_t seg[NITEMS];                // lo | hi << 8 | own_row << 16 | slot << 24
    uint16_t flags[NITEMS];
    uint16_t beg[M + 1][W + 1];
    uint32_t job_mask[M + 1][W];
    uint32_t job_seg[M + 1][W];
    uint8_t njobs[M + 1];
};

__host__ __device__ constexpr int tt_lvl_base(int M, int L) { return (L - 2) * M - (L - 1) * (L - 2) / 2; }
// row of J(i..i+L-1) in the vector record: eps_1..eps_n first, then level-major
__host__ __device__ constexpr int tt_row(int N, int i, int L)
{
    return L == 1 ? i - 1 : N + tt_lvl_base(N - 1, L) + i - 1;
}

template <int N, int W>
constexpr TileTables<N, W> make_tile_tables()
{
    TileTables<N, W> t{};
    constexpr int M = N - 1;
    int base = 0;
    for (int L = 0; L <= M; ++L) {
        t.njobs[L] = 0;
        for (int w = 0; w <= W; ++w) t.beg[L][w] = 0;
    }
    for (int L = 2; L <= M; ++L) {
        const int NC = M - L + 1;
        const int per = (L - 1) + (L - 1) * (L - 2) / 2;       // items per current
        const int cnt = NC * per;
        // pass 1: fill items (without flags), total weight
        long total = 0;
        {
            int idx = base;
            for (int i = 1; i <= NC; ++i)
                for (int la = 1; la <= L - 1; ++la) {
                    const uint32_t a = (uint32_t)tt_row(N, i, la);
                    const uint32_t y = (uint32_t)(i - 1) | (uint32_t)(i - 1 + L) << 8 |
                                       (uint32_t)tt_row(N, i, L) << 16;
                    t.items[idx].x = a | (uint32_t)tt_row(N, i + la, L - la) << 8 | (uint32_t)(i + la - 1) << 16;
                    t.items[idx].y = y;
                    ++idx;
                    total += kWeight3;
                    for (int lb = 1; lb <= L - la - 1; ++lb) {
                        t.items[idx].x = a | (uint32_t)tt_row(N, i + la, lb) << 8 |
                                         (uint32_t)tt_row(N, i + la + lb, L - la - lb) << 16 | IT_KIND4 << 24;
                        t.items[idx].y = y;
                        ++idx;
                        total += kWeight4;
                    }
                }
            total += (long)NC * kWeightFinish;
        }
        // pass 2: chunk boundaries by cumulative weight
        {
            long cum = 0;
            int w = 1;
            t.beg[L][0] = (uint16_t)base;
            for (int q = 0; q < cnt; ++q) {
                while (w < W && cum * W >= (long)w * total) {
                    t.beg[L][w] = (uint16_t)(base + q);
                    ++w;
                }
                cum += (t.items[base + q].x >> 24 & IT_KIND4) ? kWeight4 : kWeight3;
                if ((q + 1) % per == 0) cum += kWeightFinish;
            }
            while (w <= W) {
                t.beg[L][w] = (uint16_t)(base + cnt);
                ++w;
            }
        }
        // pass 3: flags, slots, gather jobs
        for (int w = 0; w < W; ++w) {
            const int b = t.beg[L][w], e = t.beg[L][w + 1];
            for (int q = b; q < e; ++q) {
                const int rel = q - base, cur = rel / per, pos = rel % per;
                uint32_t fl = t.items[q].x >> 24;
                const bool first = q == b || pos == 0;
                const bool last = q == e - 1 || pos == per - 1;
                const bool newa = first || (t.items[q].x & 255u) != (t.items[q - 1].x & 255u);
                if (first) fl |= IT_SEG_START;
                if (newa) fl |= IT_LOAD_A;
                if (L == M) fl |= IT_TOP;
                if (last) {
                    fl |= IT_SEG_END;
                    // start of this segment: max(b, first item of the current)
                    const int s0 = base + cur * per;
                    const int segb = s0 > b ? s0 : b;
                    const bool complete = segb == s0 && pos == per - 1;
                    if (complete) {
                        fl |= IT_COMPLETE;
                    } else {
                        const int slot = 2 * w + (segb == b ? 0 : 1);
                        t.items[q].y |= (uint32_t)slot << 24;
                        // register the slot with the current's gather job
                        int j = -1;
                        for (int z = 0; z < t.njobs[L]; ++z)
                            if ((t.jobs[L][z].y >> 16 & 255u) == (t.items[q].y >> 16 & 255u)) j = z;
                        if (j < 0) {
                            j = t.njobs[L]++;
                            t.jobs[L][j].x = 0;
                            t.jobs[L][j].y = t.items[q].y & 0x00ffffffu;
                        }
                        t.jobs[L][j].x |= 1u << slot;
                    }
                }
                t.items[q].x = (t.items[q].x & 0x00ffffffu) | fl << 24;
            }
        }
        base += cnt;
    }
    return t;
}

// rowbytes = D * sizeof(E); ps0 = first PS2 row; sc_u, sc_v = first scalar index of the U / V tables;
// scalbytes = 32 * sizeof(E), the distance between consecutive scalars of one lane
template <int N, int W>
constexpr TileProgram<N, W> make_tile_program(int rowbytes, int ps0, int sc_u, int sc_v, int scalbytes)
{
    const TileTables<N, W> t = make_tile_tables<N, W>();
    TileProgram<N, W> p{};
    for (int q = 0; q < TileTables<N, W>::NITEMS; ++q) {
        const uint32_t x = t.items[q].x;
        const uint32_t a = x & 255u, b = x >> 8 & 255u, c = x >> 16 & 255u, fl = x >> 24;
        p.off[q].a = a * rowbytes;
        p.off[q].b = b * rowbytes;
        p.off[q].c = ((fl & IT_KIND4) ? c : ps0 + c) * rowbytes;
        p.off[q].uv = (fl & IT_KIND4) ? 0u : (uint32_t)((sc_u + a) * scalbytes) | (uint32_t)((sc_v + b) * scalbytes) << 16;
        p.seg[q] = t.items[q].y;
        p.flags[q] = (uint16_t)fl;
    }
    for (int L = 0; L <= N - 1; ++L) {
        for (int w = 0; w <= W; ++w) p.beg[L][w] = t.beg[L][w];
        p.njobs[L] = t.njobs[L];
        for (int j = 0; j < W; ++j) {
            p.job_mask[L][j] = t.jobs[L][j].x;
            p.job_seg[L][j] = t.jobs[L][j].y;
        }
    }
    return p;
}

}  // namespace bg
