// bg_tables.cuh -- compile-time work lists for the tiled Berends-Giele kernel (bg_tile.cuh).
//
// The sums over splittings of Eq.(6) are flattened, level by level, into a
// list of ITEMS: for the current (i..j) of length L, in la-major order, the 3-gluon split
// (i..k | k+1..j), k = i+la-1, followed by the 4-gluon splits (i..k | k+1..l | l+1..j),
// l = k+lb.  The list of a level is cut into W contiguous chunks, one per warp of the tile,
// chosen by dynamic programming over a cost model of the level (pass 2 below), so the warps
// of a block stay balanced whatever the number of currents at that level.  A chunk boundary
// may fall inside a current (in front of a 3-gluon split); such a current gets its partial
// sums combined by a "gather job" after a block barrier.
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
        // pass 1: fill items (without flags)
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
                    for (int lb = 1; lb <= L - la - 1; ++lb) {
                        t.items[idx].x = a | (uint32_t)tt_row(N, i + la, lb) << 8 |
                                         (uint32_t)tt_row(N, i + la + lb, L - la - lb) << 16 | IT_KIND4 << 24;
                        t.items[idx].y = y;
                        ++idx;
                    }
                }
        }
        // pass 2: chunk boundaries.  Cuts are allowed in front of every 3-gluon split (the start of a
        // group of items that share the left factor); the contiguous partition into W chunks with
        // the smallest modelled level time is found by dynamic programming over the cut positions
        // (chunk cost = its items + start + finish or partial store of every current it touches, in
        // executed instructions), once freely and once with shared currents forbidden; the two are
        // compared by the full model (largest chunk + largest gather load, gather job j on warp j mod W).
        {
            constexpr int kI3 = 105, kI4 = 55, kStart = 35, kFin = 160, kPart = 70, kGather = 30;
            constexpr int MAXP = (M / 2 + 1) * (M / 2 + 1) + 2;
            int pos[MAXP] = {};
            int np = 0;
            for (int q = 0; q < cnt; ++q)
                if (!(t.items[base + q].x >> 24 & IT_KIND4)) pos[np++] = q;
            pos[np++] = cnt;
            long pre[MAXP] = {};                               // cost of the items before position k
            for (int k = 0; k + 1 < np; ++k) {
                long c = 0;
                for (int q = pos[k]; q < pos[k + 1]; ++q) c += (t.items[base + q].x >> 24 & IT_KIND4) ? kI4 : kI3;
                pre[k + 1] = pre[k] + c;
            }
            long best_time = -1;
            for (int cand = 0; cand < 2; ++cand) {
                const long pen = cand == 0 ? 0 : 1000000;
                long bestv[W + 1][MAXP] = {};
                int arg[W + 1][MAXP] = {};
                for (int w = 0; w <= W; ++w)
                    for (int k = 0; k < np; ++k) bestv[w][k] = (w == 0 && k == 0) ? 0 : (long)1 << 60;
                for (int w = 1; w <= W; ++w)
                    for (int k = 0; k < np; ++k)
                        for (int pk = 0; pk <= k; ++pk) {
                            if (bestv[w - 1][pk] >= bestv[w][k]) continue;
                            long c = 0;
                            if (pk < k) {
                                const int pq = pos[pk], qq = pos[k];
                                c = pre[k] - pre[pk];
                                for (int cur = pq / per; cur <= (qq - 1) / per; ++cur) {
                                    const bool whole = pq <= cur * per && qq >= (cur + 1) * per;
                                    c += kStart + (whole ? kFin : kPart + pen);
                                }
                            }
                            const long v = bestv[w - 1][pk] > c ? bestv[w - 1][pk] : c;
                            if (v < bestv[w][k]) { bestv[w][k] = v; arg[w][k] = pk; }
                        }
                int cc[W + 1] = {};
                for (int w = W, k = np - 1; w >= 1; --w) { cc[w] = pos[k]; k = arg[w][k]; }
                // full model
                long la = 0, lb = 0, gl[W] = {};
                int shared_parts[M + 1] = {};
                for (int w = 0; w < W; ++w) {
                    const int pq = cc[w], qq = cc[w + 1];
                    if (pq >= qq) continue;
                    long c = 0;
                    for (int q = pq; q < qq; ++q) c += (t.items[base + q].x >> 24 & IT_KIND4) ? kI4 : kI3;
                    for (int cur = pq / per; cur <= (qq - 1) / per; ++cur) {
                        const bool whole = pq <= cur * per && qq >= (cur + 1) * per;
                        c += kStart + (whole ? kFin : kPart);
                        if (!whole) ++shared_parts[cur];
                    }
                    if (c > la) la = c;
                }
                int nj = 0;
                for (int cur = 0; cur < NC; ++cur)
                    if (shared_parts[cur]) {
                        gl[nj % W] += kFin + (long)shared_parts[cur] * kGather;
                        if (gl[nj % W] > lb) lb = gl[nj % W];
                        ++nj;
                    }
                if (nj <= W && (best_time < 0 || la + lb < best_time)) {
                    best_time = la + lb;
                    for (int w = 0; w <= W; ++w) t.beg[L][w] = (uint16_t)(base + cc[w]);
                }
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
