// bg_reg.cuh -- register-resident Berends-Giele kernel for few gluons: every current J(i..j) of a
// point lives in REGISTERS, split over two lanes.
//
// Why: the complex128 tiled kernels are bound by shared-memory bandwidth as much as by the FP64
// pipe (a 16-byte element per lane makes every vector load four wavefronts; a 4-gluon split loads
// two vectors for 32 DFMA -- DESIGN.md §7).  For n = 6, d = 4 the 15 currents of a point are 60
// complex numbers: held as 2 components per lane in the lane pair (l, l+16) that is 120
// registers, and the whole recursion of Eq.(6) can be unrolled with compile-time
// indices so that no vector is ever loaded from shared memory.  Only the per-current scalars U, V
// and 1/P^2 and the doubled prefix sums PS2_c stay in shared memory (lane-private columns: a
// lane only reads what it wrote itself, so the kernel has NO barrier and no inter-warp
// communication at all; a warp owns 16 points from load to store).
//
// Same algebra as the tiled kernels (factored form, bg_tile.cuh); Minkowski products are the sum
// of the two lanes' partial products (bg_split.cuh).  Inputs are read straight from global memory
// into registers (32 contiguous bytes per lane and row).
#pragma once
#include <cuda_pipeline.h>

#include "bg_common.cuh"
#include "bg_schedule.cuh"

namespace bg {
template <class F, int N, int D>
struct RegCfg {
    typedef typename F::E E;
    static constexpr int M = N - 1;
    static constexpr int DL = D / 2, TP = 16;
    static constexpr int R = M * (M - 1) / 2 - 1;
    static constexpr int J_ROWS = N + R;                      // eps_1..eps_n, then multi-gluon level-major (top excluded)
    // per-warp shared memory, [index][16 points]: PS2 rows (M+1) x D components, U, V per row, W per range
    static constexpr int PS_OFF = 0;
    static constexpr int U_OFF = (M + 1) * D, V_OFF = U_OFF + J_ROWS, W_OFF = V_OFF + J_ROWS;
    static constexpr int NSCAL = W_OFF + R;
    static constexpr int WARPS = 4;                           // independent warps per block
    static constexpr int MIN_BLOCKS = 2;                      // 236 registers, no spills (3 blocks: 168 registers, 80 B of spills, same speed)
    // input staging buffer of a warp: eps_1..eps_n and k_1..k_m of its NEXT 16 points, copied with cp.async
    // while the current 16 points are computed; point stride an odd number of elements (conflict-free)
    static constexpr int IN_ROWS = N + M;
    static constexpr int IN_STRIDE = (IN_ROWS * D) | 1;
    static constexpr size_t SMEM_BYTES = (size_t)WARPS * (NSCAL + IN_STRIDE) * TP * sizeof(E);
};

// row of J(i..i+len-1), i 1-based
template <int N>
__host__ __device__ constexpr int reg_row(int i, int len) { return tt_row(N, i, len); }

// -(x.y) of two vectors held as (lane 0: components 0..DL-1, lane 1: the rest); full value in both lanes
template <class F, int MET, int DL, int TP>
__device__ __forceinline__ typename F::E reg_dot_neg(const F& f, int mu0, const typename F::E (&x)[DL],
                                                     const typename F::E (&y)[DL])
{
    typename F::E nx[DL];
    lower_neg<F, MET, DL>(f, mu0, x, nx);
    return lane_sum<F, 2, TP>(f, f.reduce(dot_plain<F, DL>(f, nx, y)));
}
template <class F, int DL, int TP>
__device__ __forceinline__ typename F::E reg_dot_plain(const F& f, const typename F::E (&x)[DL],
                                                       const typename F::E (&y)[DL])
{
    return lane_sum<F, 2, TP>(f, f.reduce(dot_plain<F, DL>(f, x, y)));
}

template <class F, int MET, int N, int D>
__global__ void __launch_bounds__(32 * RegCfg<F, N, D>::WARPS, RegCfg<F, N, D>::MIN_BLOCKS) bg_reg_kernel(const BgParams<F> prm)
{
    typedef RegCfg<F, N, D> C;
    typedef typename F::E E;
    typedef typename F::A A;
    constexpr int M = C::M, DL = C::DL, TP = C::TP, ND = N * D;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int point = lane & (TP - 1), half = lane / TP, mu0 = half * DL;
    const F f(prm.fld, 0);
    E* wbase = reinterpret_cast<E*>(smem_raw) + (size_t)warp * (C::NSCAL + C::IN_STRIDE) * TP;
    E* sc = wbase + point;                                    // [index][TP], this point's column
    E* inbuf = wbase + C::NSCAL * TP;                         // [TP][IN_STRIDE]
    // Persistent warps: warp w of the grid owns the 16-point groups w, w + (warps in the grid), ...  The inputs
    // of the next group are copied global -> shared with cp.async while the current group is computed, so the
    // HBM latency (17 % of the stall samples when the inputs went straight to registers) is off the critical path.
    const long long ngroups = (prm.batch + TP - 1) / TP;
    const long long gstep = (long long)gridDim.x * C::WARPS;
    auto prefetch = [&](long long g) {
        constexpr int CH_POL = N * D, CH = C::IN_ROWS * D;    // elements per point: eps rows, then k_1..k_m
        for (int idx = lane; idx < TP * CH; idx += 32) {
            const int p = idx / CH, w = idx - p * CH;
            long long gp = g * TP + p;
            gp = gp < prm.batch ? gp : prm.batch - 1;         // ragged last group: repeat the last point (no stores)
            const E* src = w < CH_POL ? prm.pol + gp * ND + w : prm.mom + gp * ND + (w - CH_POL);
            __pipeline_memcpy_async(inbuf + p * C::IN_STRIDE + w, src, sizeof(E));
        }
        __pipeline_commit();
    };
    long long g = (long long)blockIdx.x * C::WARPS + warp;
    if (g < ngroups) prefetch(g);
#pragma unroll 1
    for (; g < ngroups; g += gstep) {
    const long long pt = g * TP + point;
    const bool live = pt < prm.batch;

    E J[C::J_ROWS + 1][DL];                                   // + the top current
    uint32_t status = 0;

    // ---- a0/a1: eps rows into registers; doubled prefix sums PS2_c into the lane's column; U = V = 2 k.eps
    __pipeline_wait_prior(0);
    __syncwarp();
    {
        const E* gp = inbuf + point * C::IN_STRIDE + half * DL;
        const E* gm = gp + N * D;
        E run[DL];
#pragma unroll
        for (int mu = 0; mu < DL; ++mu) {
            run[mu] = f.ezero();
            sc[(C::PS_OFF + mu + half * DL) * TP] = run[mu];
        }
        E kk[M][DL];
#pragma unroll
        for (int c = 1; c <= N; ++c) {
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) J[c - 1][mu] = f.load_input(gp[(c - 1) * D + mu]);
            if (c <= M) {
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) kk[c - 1][mu] = f.dbl(f.load_input(gm[(c - 1) * D + mu]));
            }
        }
        __syncwarp();                                          // every lane has its inputs: the buffer is free
        if (g + gstep < ngroups) prefetch(g + gstep);
#pragma unroll
        for (int c = 1; c <= M; ++c) {
            const E u = f.neg(reg_dot_neg<F, MET, DL, TP>(f, mu0, kk[c - 1], J[c - 1]));       // 2 k.eps
            sc[(C::U_OFF + c - 1) * TP] = u;
            sc[(C::V_OFF + c - 1) * TP] = u;
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) {
                run[mu] = f.add(run[mu], kk[c - 1][mu]);
                sc[(C::PS_OFF + c * D + mu + half * DL) * TP] = run[mu];
            }
        }
    }

    // ---- a2-a6: level sweep, everything unrolled with compile-time row indices -----------------------
#pragma unroll
    for (int L = 2; L <= M; ++L) {
#pragma unroll
        for (int ci = 0; ci + L <= M; ++ci) {
            const int i = ci + 1;
            E l[DL], h[DL], x2[DL];
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) {
                l[mu] = sc[(C::PS_OFF + ci * D + mu + half * DL) * TP];            // PS2_{i-1}
                h[mu] = sc[(C::PS_OFF + (ci + L) * D + mu + half * DL) * TP];      // PS2_j
            }
            lower_diff<F, MET, DL>(f, mu0, h, l, x2);                                // 2 * covariant P_{i,j}
            A acc[DL];
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) acc[mu] = f.zero();
            E hsum = f.ezero();
            int room = F::kCap0;
            auto need = [&](int k) {
                if (room < k) {
#pragma unroll
                    for (int mu = 0; mu < DL; ++mu) acc[mu] = f.relief(acc[mu]);
                    room = F::kCapR;
                }
                room -= k;
            };
#pragma unroll
            for (int la = 1; la <= L - 1; ++la) {
                const int ra = reg_row<N>(i, la), rb = reg_row<N>(i + la, L - la);
                E s[DL];
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) s[mu] = sc[(C::PS_OFF + (ci + la) * D + mu + half * DL) * TP];
                const E ua = sc[(C::U_OFF + ra) * TP], vb = sc[(C::V_OFF + rb) * TP];
                const E hk = f.neg(reg_dot_neg<F, MET, DL, TP>(f, mu0, J[ra], J[rb]));    // A.B
                const E xa = reg_dot_plain<F, DL, TP>(f, x2, J[ra]);                 // 2 X.A
                const E xb = reg_dot_plain<F, DL, TP>(f, x2, J[rb]);                 // 2 X.B
                const E cb = f.sub(xa, ua);
                const E ca = f.sub(vb, xb);
                hsum = f.add(hsum, hk);
                need(2);
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) {
                    acc[mu] = f.mad(hk, s[mu], acc[mu]);
                    acc[mu] = f.mad(cb, J[rb][mu], acc[mu]);
                }
                need(1);
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) acc[mu] = f.mad(ca, J[ra][mu], acc[mu]);
#pragma unroll
                for (int lb = 1; lb <= L - la - 1; ++lb) {
                    const int rm = reg_row<N>(i + la, lb), rc = reg_row<N>(i + la + lb, L - la - lb);
                    const E cc = f.neg(f.dbl(reg_dot_neg<F, MET, DL, TP>(f, mu0, J[ra], J[rc])));   // 2 A.C
                    need(1);
#pragma unroll
                    for (int mu = 0; mu < DL; ++mu) acc[mu] = f.mad(cc, J[rm][mu], acc[mu]);
                }
            }
            // ---- finish: boundary term of the (P-Q) sum, propagator, U and V --------------------------
            const E nhh = f.neg(f.mul(hsum, f.half()));                          // -(sum_k h_k)/2
            need(2);
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) {
                acc[mu] = f.mad(nhh, l[mu], acc[mu]);
                acc[mu] = f.mad(nhh, h[mu], acc[mu]);
            }
            const int own = L < M ? reg_row<N>(i, L) : C::J_ROWS;
            if (L < M) {
                E xc[DL];
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) xc[mu] = f.sub(h[mu], l[mu]);      // 2 P_{i,j}, contravariant
                const E s4 = f.canon(f.neg(reg_dot_neg<F, MET, DL, TP>(f, mu0, xc, xc)));  // 4 P^2
                if (f.is_zero(s4)) status |= 1u;
                const E w = f.dbl(f.dbl(f.inv(s4)));                              // 1/P^2, inv(0) := 0
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) J[own][mu] = f.mul(f.reduce(acc[mu]), w);
                const E c2 = reg_dot_plain<F, DL, TP>(f, x2, J[own]);                 // 2 P_{i,j} . J(i..j)
                sc[(C::U_OFF + own) * TP] = f.add(c2, hsum);
                sc[(C::V_OFF + own) * TP] = f.sub(c2, hsum);
            } else {
                // top current: no propagator; amplitude = eps_n . N(1..m)
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) J[own][mu] = f.reduce(acc[mu]);
                const E nout = reg_dot_neg<F, MET, DL, TP>(f, mu0, J[N - 1], J[own]);
                if (live && half == 0) prm.out[pt] = f.to_output(f.neg(nout));
            }
            if (prm.currents && live) {
                E* dst = prm.currents + (pt * M * M + (long long)ci * M + (ci + L - 1)) * D + half * DL;
#pragma unroll
                for (int mu = 0; mu < DL; ++mu) dst[mu] = f.to_output(J[own][mu]);
            }
        }
    }
    if (prm.currents && live) {
#pragma unroll
        for (int c = 0; c < M; ++c) {
            E* dst = prm.currents + (pt * M * M + (long long)c * M + c) * D + half * DL;
#pragma unroll
            for (int mu = 0; mu < DL; ++mu) dst[mu] = f.to_output(J[c][mu]);
        }
    }
    if (prm.status && live && half == 0) prm.status[pt] = status;
    __syncwarp();                                              // lane-private columns are rewritten by the next group
    }
}

}  // namespace bg
