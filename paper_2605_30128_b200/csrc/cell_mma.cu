// Tensor-core cell kernel: S1 gather, S2 cell Laplacian, S3 assembly, S5 pointwise + update in one pass, with the three
// 1-D contractions of the sum-factorised Laplacian issued as warp-level matrix instructions.
//
// Why tensor instructions here (north_star kernel (2): "only if ncu shows the contraction is compute-bound"): the line-owned
// FFMA/DFMA kernel (cell_xyz.cu) is issue-bound -- profiles/r2_c3_cell_kernels.md: 62 % issue-active with 8.1 instructions
// per unit in the FP32-stored mode, 39 % with 2.7 warps per scheduler in FP64 -- so the lever is instructions per unit,
// not flops.  One mma.sync.m16n8k8.tf32 replaces 32 FFMA warp instructions, one mma.sync.m8n8k4.f64 eight DFMA ones.
// (tcgen05.mma was evaluated and rejected for this contraction: its A operand must be the data tile, M = 128 rows by
// K = 8 deep from shared memory, 4 KB per instruction for a 9-wide B; at the measured ~128 B/clk of operand bandwidth that
// is >= 32 clk per instruction, 3.9 kclk per plane and contraction pass against a 1.8 kclk HBM budget -- DESIGN.md 6.5.)
//
// Formulation.  For each direction the contraction is  D[col][out] = sum_in A[col][in] B[in][out]  with
//   A = the data (M = the CTA's real batch columns of one spin component: 16 for TF32, 8 for FP64; K = the p+1 nodes of a
//       line), loaded as fragments straight from the TMA-landed plane in shared memory,
//   B = the (p+1) x (p+1) 1-D operator, transposed, held as fragments in registers for the whole kernel.
// A CTA owns the xy-footprint of one cell column, a z-segment and C real batch columns, and marches through the planes:
//   X task (warp = row j, spin):   x-contraction of row j of plane t+1        -> shared XR (one plane ahead)
//   Y task (warp = x-position i):  y-contraction at x-position i of plane t, + XR, + S5 on owned nodes -> RED to `out`
//   Z task (at the end of a cell): z-contraction over the p+1 planes of the cell, which are all resident in the plane
//                                  ring (no z accumulators in registers), for the warp's row of nodes    -> RED to `out`
// D comes out as (column g, outputs 2t, 2t+1): eight lanes hold eight adjacent columns, so every RED covers full 32-byte
// sectors.  An output node receives two REDs (in-plane part + S5, z part) instead of one.
// Modes: MM_F64 (complex128 storage, mma.m8n8k4.f64), MM_TF32 (complex64 storage, operands rounded cvt.rna.tf32.f32, FP32
// accumulate: CHFSI_TF32), MM_TF32X3 (hi/lo split of both operands, three MMAs, small terms first: CHFSI_TF32X3).
#include <cuda.h>

#include <cstring>
#include <mutex>
#include <type_traits>

#include "chfsi_internal.h"
#include "tma_util.cuh"

namespace chfsi {

enum MmaMode : int { MM_TF32 = 0, MM_TF32X3 = 1, MM_F64 = 2 };

template <int MODE> struct MmaTraits { using T = float; static constexpr int MROWS = 16, KSTEP = 8; };
template <> struct MmaTraits<MM_F64> { using T = double; static constexpr int MROWS = 8, KSTEP = 4; };

template <typename T>
struct MmaConst {
    T K[3][kMaxN][kMaxN];       // scaled 1-D operators K[d][out][in] (all scalings folded in, see build_mma_const)
    T W[3][kMaxN];              // WX, WY, WZ
    double cHp;                 // coefficient of the potential term
};

template <int P, int MODE>
struct MmaCfg {
    using T = typename MmaTraits<MODE>::T;
    static constexpr int n = P + 1;
    static constexpr int MROWS = MmaTraits<MODE>::MROWS, KSTEP = MmaTraits<MODE>::KSTEP;
    static constexpr int C = 2 * MROWS, NV = C / 4;          // real batch columns of the CTA: both spin components
    static constexpr int NR = MROWS / 8, KH = KSTEP / 4;     // fragment rows g + 8r, fragment k-halves t + 4h
    static constexpr int KS = (n + KSTEP - 1) / KSTEP, NT = (n + 7) / 8;
    static constexpr int NCW = 2 * n;                        // consumer warps: (index q in 0..p) x (spin)
    static constexpr int THREADS = (NCW + 1) * 32;
    static constexpr int ESZ = (int)sizeof(T);
    // plane ring stage: MAIN [n lines][P nodes][C] | FACE [n lines][C] (the x = P column)
    static constexpr int FACE_ELEMS = n * P * C;
    static constexpr int IN_BYTES = n * n * C * ESZ;
    static constexpr int IN_STAGE = ((IN_BYTES + 127) / 128) * 128;
    // R / fields ring stage: R [P][P][C] f64 | fields [P][P][4] f64
    static constexpr int R_BYTES = P * P * C * 8, F_BYTES = P * P * 32;
    static constexpr int R_STAGE = ((R_BYTES + F_BYTES + 127) / 128) * 128;
    static constexpr int RS = 3;
    // XR[row][x'][XP]: the x-contraction of a plane, column pitch padded by 16 bytes (bank spread of the fragment accesses)
    static constexpr int XP = C + 16 / ESZ;
    static constexpr int XR_BYTES = ((n * n * XP * ESZ + 127) / 128) * 128;
    static constexpr int S_ = (220 * 1024 - 2 * XR_BYTES - RS * R_STAGE) / IN_STAGE;
    static constexpr int S = S_ < 16 ? S_ : 16;
    static_assert(S >= P + 2, "plane ring must hold a whole cell plus the plane ahead");
    static constexpr size_t SMEM = (size_t)S * IN_STAGE + (size_t)RS * R_STAGE + 2 * (size_t)XR_BYTES;
};

__device__ __forceinline__ void red_add_t(double* p, double v) { atomicAdd(p, v); }     // result unused -> RED
__device__ __forceinline__ void red_add_t(float* p, float v) { atomicAdd(p, v); }

__device__ __forceinline__ uint32_t to_tf32(float x) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void mma_tf32(float (&d)[2][2], const uint32_t (&a)[2][2], const uint32_t (&b)[2]) {
    // a[r][h] = A(row g + 8r, k = t + 4h) -> a0 = a[0][0], a1 = a[1][0], a2 = a[0][1], a3 = a[1][1]; d[r][e] = D(row g + 8r, col 2t + e)
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0][0]), "+f"(d[0][1]), "+f"(d[1][0]), "+f"(d[1][1])
                 : "r"(a[0][0]), "r"(a[1][0]), "r"(a[0][1]), "r"(a[1][1]), "r"(b[0]), "r"(b[1]));
}
__device__ __forceinline__ void mma_f64(double (&d)[1][2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d[0][0]), "+d"(d[0][1]) : "d"(a), "d"(b));
}

// B fragments of the three 1-D operators, per thread: B[k = in][n = out] = K[out][in]
template <int P, int MODE>
struct BFrags {
    using Cfg = MmaCfg<P, MODE>;
    using T = typename Cfg::T;
    using TB = typename std::conditional<MODE == MM_F64, double, uint32_t>::type;
    TB hi[3][Cfg::KS][Cfg::NT][Cfg::KH];
    TB lo[MODE == MM_TF32X3 ? 3 : 1][Cfg::KS][Cfg::NT][Cfg::KH];

    __device__ __forceinline__ void init(const MmaConst<T>& sc, int g, int t) {
#pragma unroll
        for (int d = 0; d < 3; ++d)
#pragma unroll
            for (int ks = 0; ks < Cfg::KS; ++ks)
#pragma unroll
                for (int nt = 0; nt < Cfg::NT; ++nt)
#pragma unroll
                    for (int h = 0; h < Cfg::KH; ++h) {
                        const int out = nt * 8 + g, in = ks * Cfg::KSTEP + t + 4 * h;
                        const T v = (out < Cfg::n && in < Cfg::n) ? sc.K[d][out < Cfg::n ? out : 0][in < Cfg::n ? in : 0] : (T)0;
                        if constexpr (MODE == MM_F64) {
                            hi[d][ks][nt][h] = v;
                        } else {
                            const uint32_t vh = to_tf32(v);
                            hi[d][ks][nt][h] = vh;
                            if constexpr (MODE == MM_TF32X3) lo[d][ks][nt][h] = to_tf32(v - __uint_as_float(vh));
                        }
                    }
    }
};

template <int P, int MODE>
struct Acc {
    using Cfg = MmaCfg<P, MODE>;
    typename Cfg::T d[Cfg::NT][Cfg::NR][2];
    __device__ __forceinline__ void zero() {
#pragma unroll
        for (int nt = 0; nt < Cfg::NT; ++nt)
#pragma unroll
            for (int r = 0; r < Cfg::NR; ++r) { d[nt][r][0] = 0; d[nt][r][1] = 0; }
    }
};

// acc += (operator of direction DIR) applied along the line whose element kk = KSTEP ks + t + 4 h (0..p) for fragment row r
// is ld(ks, h, kk, r)
template <int P, int MODE, int DIR, typename LD>
__device__ __forceinline__ void contract(Acc<P, MODE>& acc, const BFrags<P, MODE>& bf, int t, LD ld) {
    using Cfg = MmaCfg<P, MODE>;
    using T = typename Cfg::T;
#pragma unroll
    for (int ks = 0; ks < Cfg::KS; ++ks) {
        T a[Cfg::NR][Cfg::KH];
#pragma unroll
        for (int h = 0; h < Cfg::KH; ++h) {
            const int kk = ks * Cfg::KSTEP + t + 4 * h;
            // the last k-step is only partly populated: lanes beyond the line contribute zeros
            const bool ok = (ks * Cfg::KSTEP + 3 + 4 * h < Cfg::n) || kk < Cfg::n;
#pragma unroll
            for (int r = 0; r < Cfg::NR; ++r) a[r][h] = ok ? ld(ks, h, kk, r) : (T)0;
        }
        if constexpr (MODE == MM_F64) {
#pragma unroll
            for (int nt = 0; nt < Cfg::NT; ++nt) mma_f64(acc.d[nt], a[0][0], bf.hi[DIR][ks][nt][0]);
        } else {
            uint32_t ah[2][2], al[2][2];
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    ah[r][h] = to_tf32(a[r][h]);
                    if constexpr (MODE == MM_TF32X3) al[r][h] = to_tf32(a[r][h] - __uint_as_float(ah[r][h]));
                }
#pragma unroll
            for (int nt = 0; nt < Cfg::NT; ++nt) {
                if constexpr (MODE == MM_TF32X3) {
                    mma_tf32(acc.d[nt], al, bf.hi[DIR][ks][nt]);       // small terms first
                    mma_tf32(acc.d[nt], ah, bf.lo[DIR][ks][nt]);
                }
                mma_tf32(acc.d[nt], ah, bf.hi[DIR][ks][nt]);
            }
        }
    }
}

template <int P, int MODE, bool HASPH>
__global__ void __launch_bounds__(MmaCfg<P, MODE>::THREADS, 1)
cell_mma_kernel(const __grid_constant__ MmaConst<typename MmaCfg<P, MODE>::T> sc, const __grid_constant__ MarchArgs ar,
                const __grid_constant__ MarchMaps mp) {
    using Cfg = MmaCfg<P, MODE>;
    using T = typename Cfg::T;
    constexpr int n = Cfg::n, C = Cfg::C, S = Cfg::S, RS = Cfg::RS, XP = Cfg::XP, NR = Cfg::NR, NT = Cfg::NT, MROWS = Cfg::MROWS;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full_in[S], empty_in[S], full_r[RS], empty_r[RS];
    unsigned char* rring = smem + (size_t)S * Cfg::IN_STAGE;
    T* XRb = reinterpret_cast<T*>(rring + (size_t)RS * Cfg::R_STAGE);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int ROWB = (C / 2) * Cfg::ESZ;
    constexpr int PAIR = ROWB >= 128 ? 1 : 128 / ROWB;
    int bid = blockIdx.x;
    const int cpair = bid % PAIR; bid /= PAIR;
    const int ex = bid % ar.nc[0]; bid /= ar.nc[0];
    const int ey = bid % ar.nc[1]; bid /= ar.nc[1];
    const int seg = bid % ar.nseg;
    const int chunk = PAIR * (bid / ar.nseg) + cpair;
    if (chunk >= ar.nchunks) return;
    const int T_ = ar.cps * P + 1;                // planes this CTA marches through
    const int g0 = seg * ar.cps * P;              // first global plane
    const bool xwrap = ex == ar.nc[0] - 1, ywrap = ey == ar.nc[1] - 1;

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full_in[s], 1); mbar_init(&empty_in[s], Cfg::NCW); }
        for (int s = 0; s < RS; ++s) { mbar_init(&full_r[s], 1); mbar_init(&empty_r[s], Cfg::NCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == Cfg::NCW) {
        // ================================ producer (S1 gather, PAPER.md:204 (i)) ================================
        if (lane == 0) {
            const int col0 = chunk * (C / 2);
            uint64_t pol_last;
            asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_last));
            for (int t = 0; t < T_; ++t) {
                const int s = t % S;
                mbar_wait(&empty_in[s], ((t / S) & 1) ^ 1);
                mbar_expect_tx(&full_in[s], Cfg::IN_BYTES);
                unsigned char* st = smem + (size_t)s * Cfg::IN_STAGE;
                int gz = g0 + t; if (gz == ar.n1[2]) gz = 0;
                const int line = gz * ar.n1[1] + ey * P;
                const int xr = 2 * ex * P;
                const int xf = xwrap ? 0 : xr + 2 * P;
                if (!ywrap) {
                    tma_load_3d(st, &mp.main[0], col0, xr, line, &full_in[s]);
                    tma_load_3d(st + Cfg::FACE_ELEMS * Cfg::ESZ, &mp.face[0], col0, xf, line, &full_in[s]);
                } else {
                    tma_load_3d(st, &mp.main[1], col0, xr, line, &full_in[s]);
                    tma_load_3d(st + P * P * C * Cfg::ESZ, &mp.main[2], col0, xr, gz * ar.n1[1], &full_in[s]);
                    tma_load_3d(st + Cfg::FACE_ELEMS * Cfg::ESZ, &mp.face[1], col0, xf, line, &full_in[s]);
                    tma_load_3d(st + (Cfg::FACE_ELEMS + P * C) * Cfg::ESZ, &mp.face[2], col0, xf, gz * ar.n1[1], &full_in[s]);
                }
                if (t < T_ - 1) {                              // owned plane: R and the packed fields for S5
                    const int rs = t % RS;
                    mbar_wait(&empty_r[rs], ((t / RS) & 1) ^ 1);
                    mbar_expect_tx(&full_r[rs], Cfg::F_BYTES + (ar.useR ? Cfg::R_BYTES : 0));
                    unsigned char* rt = rring + (size_t)rs * Cfg::R_STAGE;
                    if (ar.useR) tma_load_3d(rt, &mp.R, chunk * (C / 2), xr, line, &full_r[rs]);
                    tma_load_2d_hint(rt + Cfg::R_BYTES, &mp.F, 4 * ex * P, line, &full_r[rs], pol_last);
                }
            }
        }
        return;
    }

    // ================================ consumers ================================
    const int mt = warp & 1, q = warp >> 1;       // spin component (= m-tile), index: row j (X, Z tasks) / x-position i (Y task)
    const int g = lane >> 2, t4 = lane & 3;
    const int col0 = mt * MROWS + g;              // fragment row r is column col0 + 8 r
    const int ri = g & 1;
    const double sg = ((ri == 0) != (mt == 0)) ? -1.0 : 1.0;
    BFrags<P, MODE> bf;
    bf.init(sc, g, t4);
    bool vok[NR];
    double cin[NR], cR[NR];
    long long ocol[NR];                           // scalar offset of the thread's column inside a node's 4 ld scalars
#pragma unroll
    for (int r = 0; r < NR; ++r) {
        const int vl = (8 * r + g) >> 1;
        const int v = chunk * Cfg::NV + vl;
        vok[r] = v < ar.nvec;
        cin[r] = (vok[r] && ar.cin) ? __ldg(ar.cin + v) : 0.0;
        cR[r] = (vok[r] && ar.cR && ar.useR) ? __ldg(ar.cR + v) : 0.0;
        ocol[r] = ((long long)mt * ar.ld_out + (vok[r] ? v : 0)) * 2 + ri;
    }
    const long long XS = 4 * ar.ld_out, LS = (long long)ar.n1[0] * XS, PS = (long long)ar.n1[1] * LS;
    T* const outp = reinterpret_cast<T*>(ar.out);
    const bool xph = HASPH && xwrap && ar.phd[0], yph = HASPH && ywrap && ar.phd[1];
    const T WXq = sc.W[0][q], WYq = sc.W[1][q];
    // node offsets of the footprint: x-position i / line j of this cell column, wrapped
    auto xoff = [&](int i) { int gx = ex * P + i; if (gx == ar.n1[0]) gx = 0; return (long long)gx * XS; };
    auto yoff = [&](int j) { int gy = ey * P + j; if (gy == ar.n1[1]) gy = 0; return (long long)gy * LS; };
    auto zoff = [&](int gzp) { if (gzp == ar.n1[2]) gzp = 0; return (long long)gzp * PS; };
    auto stage = [&](int tp) { return reinterpret_cast<T*>(smem + (size_t)(tp % S) * Cfg::IN_STAGE); };
    const int NTH = Cfg::NCW * 32;

    // conj(phase) on a wrapped output: own' = own pr + (ri ? -other pi : other pi), the partner component sits in lane ^ 4
    auto conj_phase = [&](T val, double pr, double pi) {
        const T other = __shfl_xor_sync(0xffffffffu, val, 4);
        return (T)fma((double)other, ri ? -pi : pi, (double)val * pr);
    };

    // ---- X task of plane tp: x-contraction of row q -> XR[tp & 1]
    auto xtask = [&](int tp) {
        T* IN = stage(tp);
        if (HASPH) {
            // Bloch phase on wrapped entries of the landed plane (x: the face column; y: row P; z: the whole wrapped plane),
            // fixed up in place before any task reads the plane (boundary CTAs only); this warp fixes row q of its spin
            const bool wz = ar.phd[2] && (g0 + tp) == ar.n1[2];
            if (xph | yph | wz) {                                       // CTA-uniform
                double br = 1.0, bi = 0.0;
                if (yph && q == P) { br = ar.ph_re[1]; bi = ar.ph_im[1]; }
                if (wz) { const double u = br * ar.ph_re[2] - bi * ar.ph_im[2]; bi = br * ar.ph_im[2] + bi * ar.ph_re[2]; br = u; }
                const bool rowph = (yph && q == P) || wz;
                for (int i0 = 0; i0 < n; i0 += 4) {                     // lanes t4 share the row's nodes; uniform trip count (shuffles)
                    const int i = i0 + t4;
                    const bool valid = i < n;
                    double pr = br, pi = bi;
                    const bool fx = i == P && xph;
                    if (fx) { const double u = pr * ar.ph_re[0] - pi * ar.ph_im[0]; pi = pr * ar.ph_im[0] + pi * ar.ph_re[0]; pr = u; }
                    T* e = IN + (i < P ? (q * P + i) * C : Cfg::FACE_ELEMS + q * C) + col0;
#pragma unroll
                    for (int r = 0; r < NR; ++r) {
                        const T val = valid ? e[8 * r] : (T)0;
                        const T other = __shfl_xor_sync(0xffffffffu, val, 4);
                        if (valid && (rowph || fx)) e[8 * r] = (T)fma((double)other, ri ? pi : -pi, (double)val * pr);
                    }
                }
                // these stage bytes are later rewritten by TMA.  No barrier here: this warp's X task reads only the row it
                // fixed; every other reader of the plane (Y and Z tasks) runs after the barrier that ends the step.
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
            }
        }
        Acc<P, MODE> acc;
        acc.zero();
        const T* mainp = IN + (q * P) * C + col0;
        const T* facep = IN + Cfg::FACE_ELEMS + q * C + col0;
        contract<P, MODE, 0>(acc, bf, t4, [&](int, int, int kk, int r) { return kk < P ? mainp[kk * C + 8 * r] : facep[8 * r]; });
        T* XR = XRb + (size_t)(tp & 1) * (Cfg::XR_BYTES / Cfg::ESZ) + (q * n) * XP + col0;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int xo = nt * 8 + 2 * t4 + e;
                if (nt * 8 + 6 + e < n || xo < n) {
#pragma unroll
                    for (int r = 0; r < NR; ++r) XR[xo * XP + 8 * r] = WYq * acc.d[nt][r][e];
                }
            }
    };

    // ---- Y task of plane tp: y-contraction at x-position q, + XR, + S5 on owned nodes, RED to out (S3 + S5)
    auto ytask = [&](int tp, int c, bool lower, bool upper) {
        const T* IN = stage(tp);
        const int rs = tp % RS;
        const double* Rs = reinterpret_cast<const double*>(rring + (size_t)rs * Cfg::R_STAGE);
        const double* Fs = reinterpret_cast<const double*>(rring + (size_t)rs * Cfg::R_STAGE + Cfg::R_BYTES);
        Acc<P, MODE> acc;
        acc.zero();
        const T* base = IN + (q < P ? q * C : Cfg::FACE_ELEMS) + col0;
        const int stride = q < P ? P * C : C;
        contract<P, MODE, 1>(acc, bf, t4, [&](int, int, int kk, int r) { return base[kk * stride + 8 * r]; });
        const T* XR = XRb + (size_t)(tp & 1) * (Cfg::XR_BYTES / Cfg::ESZ) + q * XP + col0;
        // the plane's in-plane part belongs to the cell above (weight W_z[c]) and, on a cell boundary, to the cell below (W_z[P])
        const T wz = (upper ? sc.W[2][c] : (T)0) + (lower ? sc.W[2][P] : (T)0);
        const bool zwrap = (g0 + tp) == ar.n1[2];
        const bool zp = HASPH && zwrap && ar.phd[2];
        const bool anyph = HASPH && ((q == P && xph) || yph || zp);    // warp-uniform
        double pr0 = 1.0, pi0 = 0.0, pr1 = 1.0, pi1 = 0.0;              // conj phase of rows < P / of row P (y-wrap)
        if (anyph) {
            if (q == P && xph) { pr0 = ar.ph_re[0]; pi0 = ar.ph_im[0]; }
            if (zp) { const double u = pr0 * ar.ph_re[2] - pi0 * ar.ph_im[2]; pi0 = pr0 * ar.ph_im[2] + pi0 * ar.ph_re[2]; pr0 = u; }
            pr1 = pr0; pi1 = pi0;
            if (yph) { pr1 = pr0 * ar.ph_re[1] - pi0 * ar.ph_im[1]; pi1 = pr0 * ar.ph_im[1] + pi0 * ar.ph_re[1]; }
        }
        if (upper && q < P) mbar_wait(&full_r[rs], (tp / RS) & 1);
        T* const pbase = outp + zoff(g0 + tp) + xoff(q);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int yo = nt * 8 + 2 * t4 + e;
                const bool live = nt * 8 + 6 + e < n || yo < n;          // compile-time true for fully populated n-tiles
                if (nt * 8 + e >= n) continue;                           // nothing in this fragment column at all
                const int yoc = live ? yo : 0;
                const long long yo_off = yoff(yoc);
#pragma unroll
                for (int r = 0; r < NR; ++r) {
                    T val = wz * fma(WXq, acc.d[nt][r][e], XR[(yoc * n) * XP + 8 * r]);
                    if (upper && q < P && live && yoc < P) {
                        // S5 on an owned node: eq. 12 spin blocks, in-term, R-term
                        const int o = (yoc * P + q) * C + col0 + 8 * r;
                        const double own = (double)IN[o];
                        const double osame = (double)IN[o + ((col0 ^ MROWS) - col0)];
                        const double oflip = (double)IN[o + ((col0 ^ MROWS ^ 1) - col0)];
                        const double* f = Fs + (yoc * P + q) * 4;
                        const double pot = fma(f[mt], own, fma(f[2], osame, (sg * f[3]) * oflip));
                        double s5 = fma(cin[r], own, sc.cHp * pot);
                        if (ar.useR) s5 = fma(cR[r], Rs[o], s5);
                        val += (T)s5;
                    }
                    if (anyph) val = conj_phase(val, yoc == P ? pr1 : pr0, yoc == P ? pi1 : pi0);
                    if (live && vok[r]) red_add_t(pbase + yo_off + ocol[r], val);
                }
            }
        if (upper) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_r[rs]);
        }
    };

    // ---- Z task of the cell whose planes are tb .. tb + P: z-contraction for the nodes of row q, RED to out
    auto ztask = [&](int tb) {
        // this lane's planes kk = t4 + 4 h (+ KSTEP ks): element pointers into the ring
        const T* pl[Cfg::KS][Cfg::KH];
#pragma unroll
        for (int ks = 0; ks < Cfg::KS; ++ks)
#pragma unroll
            for (int h = 0; h < Cfg::KH; ++h) {
                const int kk = ks * Cfg::KSTEP + t4 + 4 * h;
                pl[ks][h] = stage(tb + (kk < n ? kk : 0)) + col0;
            }
        const bool zwrap = (g0 + tb + P) == ar.n1[2];
        const bool zp = HASPH && zwrap && ar.phd[2];
        T* const rowbase = outp + yoff(q);
        for (int i = 0; i < n; ++i) {
            const int noff = i < P ? (q * P + i) * C : Cfg::FACE_ELEMS + q * C;
            Acc<P, MODE> acc;
            acc.zero();
            contract<P, MODE, 2>(acc, bf, t4, [&](int ks, int h, int, int r) { return pl[ks][h][noff + 8 * r]; });
            const T w = sc.W[0][i] * WYq;
            const bool anyph = HASPH && ((i == P && xph) || (q == P && yph) || zp);
            double pr0 = 1.0, pi0 = 0.0, pr1 = 1.0, pi1 = 0.0;          // conj phase of planes < P / of the wrapped top plane
            if (anyph) {
                if (i == P && xph) { pr0 = ar.ph_re[0]; pi0 = ar.ph_im[0]; }
                if (q == P && yph) { const double u = pr0 * ar.ph_re[1] - pi0 * ar.ph_im[1]; pi0 = pr0 * ar.ph_im[1] + pi0 * ar.ph_re[1]; pr0 = u; }
                pr1 = pr0; pi1 = pi0;
                if (zp) { pr1 = pr0 * ar.ph_re[2] - pi0 * ar.ph_im[2]; pi1 = pr0 * ar.ph_im[2] + pi0 * ar.ph_re[2]; }
            }
            T* const nb = rowbase + xoff(i);
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int ko = nt * 8 + 2 * t4 + e;
                    const bool live = nt * 8 + 6 + e < n || ko < n;
                    if (nt * 8 + e >= n) continue;
                    const int koc = live ? ko : 0;
                    const long long zo = zoff(g0 + tb + koc);
#pragma unroll
                    for (int r = 0; r < NR; ++r) {
                        T val = w * acc.d[nt][r][e];
                        if (anyph) val = conj_phase(val, koc == P ? pr1 : pr0, koc == P ? pi1 : pi0);
                        if (live && vok[r]) red_add_t(nb + zo + ocol[r], val);
                    }
                }
        }
    };

    // ---- march
    mbar_wait(&full_in[0], 0);
    xtask(0);
    asm volatile("bar.sync 1, %0;" ::"r"(NTH) : "memory");
    int c = 0;
#pragma unroll 1
    for (int t = 0; t < T_; ++t) {
        const bool lower = c == 0 && t > 0, upper = t < T_ - 1;
        if (upper) {
            mbar_wait(&full_in[(t + 1) % S], ((t + 1) / S) & 1);
            xtask(t + 1);                         // XR[(t+1)&1] was last read in the Y task of plane t-1, before the last barrier
        }
        ytask(t, c, lower, upper);
        if (lower) {
            ztask(t - P);                         // the cell below is complete and all its planes are still resident
            __syncwarp();
            if (lane == 0)
                for (int k = t - P; k < t; ++k) mbar_arrive(&empty_in[k % S]);     // its planes but the shared top one
        }
        asm volatile("bar.sync 1, %0;" ::"r"(NTH) : "memory");
        c = (c + 1 == P) ? 0 : c + 1;
    }
}

// ---------------------------------------------------------------------------------------------
// All scalings (1/2, Jacobian, D^-1 on the way in, M^-1 on the way out, the step coefficient) folded into the 1-D tables.
template <typename T>
static void build_mma_const(const chfsi_mesh* m, const CellArgs& a, MmaConst<T>& sc) {
    const MeshConst& mc = m->mc;
    const int n = mc.n;
    const bool sin_ = (a.flags & kScaleIn) != 0, sout_ = (a.flags & kSoutInvM) != 0;
    std::memset(&sc, 0, sizeof(sc));
    sc.cHp = a.cH;
    for (int d = 0; d < 3; ++d)
        for (int i = 0; i < n; ++i) {
            const double si = sin_ ? mc.im1[d][i] : 1.0, so = sout_ ? mc.im1[d][i] : 1.0;
            for (int b = 0; b < n; ++b) {
                const double sb = sin_ ? mc.im1[d][b] : 1.0;
                // the step coefficient rides on the x-direction factors: on K_x for the x part and on W_x for the y and z parts
                sc.K[d][i][b] = (T)((d == 0 ? a.cH : 1.0) * so * mc.Kd[d][i][b] * sb);
            }
            sc.W[d][i] = (T)((d == 0 ? a.cH : 1.0) * mc.w[i] * so * si);
        }
}

static std::once_flag g_mma_attr_once[4][3][2][32];   // [p/2 - 1][mode][phase][device]

template <int P, int MODE>
static cudaError_t launch_mma_t(const chfsi_mesh* m, const CellArgs& a, cudaStream_t st) {
    using Cfg = MmaCfg<P, MODE>;
    using T = typename Cfg::T;
    MmaConst<T> sc;
    build_mma_const<T>(m, a, sc);
    MarchArgs ar;
    std::memset(&ar, 0, sizeof(ar));
    for (int d = 0; d < 3; ++d) {
        ar.nc[d] = m->mc.nc[d]; ar.n1[d] = m->mc.n1[d];
        ar.ph_re[d] = m->mc.ph_re[d]; ar.ph_im[d] = m->mc.ph_im[d];
        ar.phd[d] = (m->mc.ph_re[d] != 1.0 || m->mc.ph_im[d] != 0.0) ? 1 : 0;
    }
    ar.has_phase = m->mc.has_phase;
    ar.nvec = a.nvec; ar.nchunks = (a.nvec + Cfg::NV - 1) / Cfg::NV;
    ar.useR = (a.R != nullptr && a.cR != nullptr) ? 1 : 0;
    ar.fields = m->dF; ar.cin = a.cin; ar.cR = a.cR; ar.out = a.out; ar.ld_out = a.ld_out;
    const long long base = (long long)ar.nc[0] * ar.nc[1] * ar.nchunks;
    int nseg = 1;
    for (int cand = 1; cand <= ar.nc[2]; ++cand)
        if (ar.nc[2] % cand == 0) { nseg = cand; if (base * cand >= 4 * 148) break; }
    ar.nseg = nseg; ar.cps = ar.nc[2] / nseg;
    MarchMaps mp;
    constexpr int BC = Cfg::C / 2;
    constexpr bool f32 = sizeof(T) == 4;
    const int nl[3] = {P + 1, P, 1};
    for (int i = 0; i < 3; ++i)
        if (!make_map3(&mp.main[i], m, a.in, a.ld_in, a.nvec, BC, 2 * P, nl[i], f32) ||
            !make_map3(&mp.face[i], m, a.in, a.ld_in, a.nvec, BC, 2, nl[i], f32))
            return cudaErrorInvalidValue;
    if (!make_map3(&mp.R, m, ar.useR ? a.R : a.in, ar.useR ? a.ld_R : a.ld_in, a.nvec, BC, 2 * P, P, ar.useR ? false : f32) ||
        !make_mapF(&mp.F, m, P))
        return cudaErrorInvalidValue;
    if (a.flags & kMassIn) return cudaErrorInvalidValue;             // the residual S0 runs on the line-owned FP64 kernel
    const bool ph = m->mc.has_phase != 0;
    auto kern = ph ? cell_mma_kernel<P, MODE, true> : cell_mma_kernel<P, MODE, false>;
    cudaError_t attr_err = cudaSuccess;
    std::call_once(g_mma_attr_once[P / 2 - 1][MODE][ph ? 1 : 0][m->device & 31], [&] {
        attr_err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
    });
    if (attr_err != cudaSuccess) return attr_err;
    constexpr int ROWB = (Cfg::C / 2) * (int)sizeof(T);
    constexpr int PAIR = ROWB >= 128 ? 1 : 128 / ROWB;
    const long long grid = (long long)ar.nc[0] * ar.nc[1] * nseg * PAIR * ((ar.nchunks + PAIR - 1) / PAIR);
    kern<<<(unsigned)grid, Cfg::THREADS, Cfg::SMEM, st>>>(sc, ar, mp);
    return cudaGetLastError();
}

bool mma_supported(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a) {
    if (prec != CHFSI_FP64 && prec != CHFSI_TF32 && prec != CHFSI_TF32X3) return false;
    if ((prec != CHFSI_FP64) != (a.store_f32 != 0)) return false;
    if (m->p != 2 && m->p != 4 && m->p != 6 && m->p != 8) return false;
    if (m->dF == nullptr || (a.flags & kMassIn)) return false;
    if (2 * m->nnodes >= (1ll << 31)) return false;
    if (a.store_f32 && ((a.ld_in & 1) || (a.ld_out & 1))) return false;
    if (((uintptr_t)a.in & 15) || ((uintptr_t)a.out & 15) || (a.R && ((uintptr_t)a.R & 15))) return false;
    return get_encode() != nullptr;
}

cudaError_t launch_cell_mma(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t st) {
#define MMA_CASE(PP)                                                                  \
    case PP:                                                                          \
        return prec == CHFSI_FP64 ? launch_mma_t<PP, MM_F64>(m, a, st)                \
             : prec == CHFSI_TF32 ? launch_mma_t<PP, MM_TF32>(m, a, st)               \
                                  : launch_mma_t<PP, MM_TF32X3>(m, a, st);
    switch (m->p) {
        MMA_CASE(2)
        MMA_CASE(4)
        MMA_CASE(6)
        MMA_CASE(8)
        default: return cudaErrorInvalidValue;
    }
#undef MMA_CASE
}

}  // namespace chfsi
