// Tensor-core cell kernel: S1 gather, S2 cell Laplacian, S3 assembly, S5 pointwise + update in one pass, with the three
// 1-D contractions of the sum-factorised Laplacian issued as warp-level matrix instructions.
//
// Why tensor instructions here (north_star kernel (2): "only if ncu shows the contraction is compute-bound"): the line-owned
// FFMA/DFMA kernel (cell_xyz.cu) is issue-bound -- profiles/r2_c3_cell_kernels.md: 62 % issue-active with 8.1 instructions
// per unit in the FP32-stored mode, 39 % with 2.7 warps per scheduler in FP64 -- so the lever is instructions per unit,
// not flops.  One mma.sync.m16n8k8.tf32 replaces 32 FFMA warp instructions, one mma.sync.m8n8k4.f64 eight DFMA ones.
// (tcgen05.mma was evaluated and rejected for this contraction: its A operand must be the data tile, M = 128 rows by
// K = 8 deep from shared memory, 4 KB per instruction for a 9-wide B; at ~128 B/clk of operand bandwidth that is >= 32 clk
// per instruction, 3.9 kclk per plane and contraction pass against a 1.8 kclk HBM budget -- DESIGN.md 6.5.)
//
// Formulation.  For each direction the contraction is  D[col][out] = sum_in A[col][in] B[in][out]  with
//   A = the data (M = the CTA's real batch columns of one spin component: 16 for TF32, 8 for FP64; K = the p+1 nodes of a
//       line), loaded as fragments straight from the TMA-landed plane in shared memory,
//   B = ONE (p+1) x (p+1) matrix for all three directions (on this mesh the scaled 1-D operators differ by a scalar),
//       transposed, held as fragments in registers for the whole kernel.
// A CTA owns the xy-footprint of one cell column, a z-segment and C real batch columns, and marches through the planes:
//   X task (warp = row j, spin):   x-contraction of row j of plane t+1, + S5 on owned nodes   -> shared XR (one plane ahead)
//   Y task (warp = x-position i):  y-contraction at x-position i of plane t, + XR             -> RED to `out`
//   Z task (at the end of a cell): z-contraction over the p+1 planes of the cell, which are all resident in the plane
//                                  ring (no z accumulators in registers), for the warp's row of nodes -> RED to `out`
// Fragment rows are chosen so that a thread's 8-byte unit of a node's 128-byte row -- one complex64 (TF32: rows g and g+8 of
// the m16 tile are its real and imaginary part) or one double (FP64) -- is: bit 3 = g & 1, bit 6 (the spin component) =
// (g >> 1) & 1, the 16-byte chunk = 2 mt + (g >> 2).  A half-warp then reads 16 distinct 8-byte slots of every landed row,
// D comes out as complex values per thread (TF32: one red.global.add.v2.f32 per output), and the lanes of a RED cover
// full 32-byte sectors.  An output node receives two REDs (in-plane part + S5, z part) instead of one.
// Shared-memory layout: a plane is [p+1 lines][p+1 nodes][2 spins][64 B] (the x = P face column sits inline as node P of its
// line), landed by TMA with the 64-byte swizzle (16-byte chunk index ^= 128-byte row index mod 4): the four k-lanes of a
// fragment load differ in node, line or plane, i.e. in the row index mod 4 (rows per line and per plane are odd, the ring has
// a multiple of 4 slots), so every fragment load is bank-conflict free.
// Modes: MM_F64 (complex128 storage, mma.m8n8k4.f64), MM_TF32 (complex64 storage, operands rounded to TF32 by
// round-to-nearest-away, FP32 accumulate: CHFSI_TF32), MM_TF32X3 (hi/lo split of both operands, three MMAs, small terms
// first: CHFSI_TF32X3).
#include <cuda.h>

#include <cmath>
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
    T K[kMaxN][kMaxN];          // base 1-D operator K[out][in]: the z-direction operator with its scalings folded in
    T W[3][kMaxN];              // WX, WY, WZ
    T sdir[3];                  // operator of direction d = sdir[d] * K   (sdir[2] = 1)
    double cHp;                 // coefficient of the potential term
};

constexpr bool kSwizzle = true;  // TMA swizzle of the plane and R stages (false: linear layout, for debugging)

template <int P, int MODE>
struct MmaCfg {
    using T = typename MmaTraits<MODE>::T;
    static constexpr int n = P + 1;
    static constexpr int MROWS = MmaTraits<MODE>::MROWS, KSTEP = MmaTraits<MODE>::KSTEP;
    static constexpr int C = 2 * MROWS, NV = C / 4;          // real batch columns of the CTA: both spin components
    static constexpr int NR = MROWS / 8, KH = KSTEP / 4;     // fragment rows g + 8r, fragment k-halves
    static constexpr int KS = (n + KSTEP - 1) / KSTEP, NT = (n + 7) / 8;
    // m-tiles per consumer warp.  2: one warp per index q running both halves of the CTA's vectors (9 warps at p = 8, ~140
    // registers, 2.56e9 warp instructions per configs[3] launch, 6.3 ms); 1: one warp per (q, m-tile) (18 warps, 96 registers).
    static constexpr int MTW = P >= 8 ? 2 : 1;       // measured: configs[3] (p = 8) 6.4 vs 6.9 ms, configs[4] (p = 6) 7.5 vs 7.2 ms
    static constexpr int NCW = n * (2 / MTW);                // consumer warps
    static constexpr int THREADS = (NCW + 1) * 32;
    static constexpr int ESZ = (int)sizeof(T);
    static_assert(C * ESZ == 128, "one node of the CTA's columns is one 128-byte row");
    // plane ring stage: [n lines][n nodes][128 B]; n is odd, so a line and a plane are an odd number of 128-byte rows
    static constexpr int LINE_BYTES = n * 128;
    static constexpr int IN_BYTES = n * n * 128;
    static constexpr int IN_STAGE = IN_BYTES;
    static_assert(n % 2 == 1, "even degrees only");
    // R / fields ring stage: R [P lines][P nodes][2 spins][C/2 doubles] | fields [P][P][4] f64
    static constexpr int R_BYTES = P * P * C * 8, F_BYTES = P * P * 32;
    static constexpr int R_STAGE = ((R_BYTES + F_BYTES + 1023) / 1024) * 1024;
    static constexpr int RS = 3;
    // XR[row][x'][XPU units of 8 bytes]: the x-contraction of a plane; 16 units per node + 1 of padding (bank spread)
    static constexpr int XPU = 17;
    static constexpr int XR_BYTES = ((n * n * XPU * 8 + 127) / 128) * 128;
    static constexpr int S_ = ((219 * 1024 - 2 * XR_BYTES - RS * R_STAGE) / IN_STAGE) / 4 * 4;     // a multiple of 4 slots
    static constexpr int S = S_ < 16 ? S_ : 16;
    static_assert(S >= P + 2, "plane ring must hold a whole cell plus the plane ahead");
    static constexpr int R_OFF = ((S * IN_STAGE + 1023) / 1024) * 1024;
    static constexpr int XR_OFF = R_OFF + RS * R_STAGE;
    static constexpr size_t SMEM = (size_t)XR_OFF + 2 * (size_t)XR_BYTES + 1024;   // + slack to align the base to 1024 B
};

// byte offset (from the 1024-aligned base) -> swizzled byte offset, as TMA lays the bytes out (measured on the B200 with a
// probe kernel: the pattern is a function of the absolute shared-memory address):
//   CU_TENSOR_MAP_SWIZZLE_64B : 16-byte chunk index bits 4..5 ^= 128-byte row index bits 7..8, rows of 64 bytes stay dense
//   CU_TENSOR_MAP_SWIZZLE_128B: chunk index bits 4..6 ^= row index bits 7..9 (used where the box rows are 128 bytes)
__device__ __forceinline__ uint32_t swz64(uint32_t lin) { return kSwizzle ? lin ^ ((lin >> 3) & 0x30u) : lin; }
__device__ __forceinline__ uint32_t swz128(uint32_t lin) { return kSwizzle ? lin ^ ((lin >> 3) & 0x70u) : lin; }

__device__ __forceinline__ void red_add_t(double* p, double v) { atomicAdd(p, v); }     // result unused -> RED
__device__ __forceinline__ void red_add_c64(float* p, float re, float im) {             // one complex64: 8-byte vector RED
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(re), "f"(im));      // `out` is never read by this kernel
}

// round-to-nearest, ties away from zero, to the 10-bit TF32 mantissa (what cvt.rna.tf32.f32 returns for finite inputs):
// add half an ulp of TF32 to the magnitude bits; the tensor core ignores the low 13 bits
__device__ __forceinline__ uint32_t to_tf32(float x) { return __float_as_uint(x) + 0x1000u; }
__device__ __forceinline__ float tf32_value(uint32_t b) { return __uint_as_float(b & 0xffffe000u); }

__device__ __forceinline__ void mma_tf32(float (&d)[2][2], const uint32_t (&a)[2][2], const uint32_t (&b)[2]) {
    // a[r][h] = A(row g + 8r, k-half h) -> a0 = a[0][0], a1 = a[1][0], a2 = a[0][1], a3 = a[1][1]; d[r][e] = D(row g + 8r, col 2t + e)
    asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0][0]), "+f"(d[0][1]), "+f"(d[1][0]), "+f"(d[1][1])
                 : "r"(a[0][0]), "r"(a[1][0]), "r"(a[0][1]), "r"(a[1][1]), "r"(b[0]), "r"(b[1]));
}
__device__ __forceinline__ void mma_f64(double (&d)[1][2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d[0][0]), "+d"(d[0][1]) : "d"(a), "d"(b));
}

// The line index that fragment position (k-step ks, half h, lane t) contracts over: the four lanes of a load read four
// consecutive nodes / lines / planes, whose 128-byte row indices differ mod 4.
template <int MODE>
__device__ __forceinline__ int kmap(int ks, int h, int t) {
    return MODE == MM_F64 ? ks * 4 + t : ks * 8 + t + 4 * h;
}

// B fragments of the base 1-D operator, per thread: B[k = in][n = out] = K[out][in]
template <int P, int MODE>
struct BFrags {
    using Cfg = MmaCfg<P, MODE>;
    using T = typename Cfg::T;
    using TB = typename std::conditional<MODE == MM_F64, double, uint32_t>::type;
    TB hi[Cfg::KS][Cfg::NT][Cfg::KH];
    TB lo[MODE == MM_TF32X3 ? Cfg::KS : 1][Cfg::NT][Cfg::KH];

    __device__ __forceinline__ void init(const MmaConst<T>& sc, int g, int t) {
#pragma unroll
        for (int ks = 0; ks < Cfg::KS; ++ks)
#pragma unroll
            for (int nt = 0; nt < Cfg::NT; ++nt)
#pragma unroll
                for (int h = 0; h < Cfg::KH; ++h) {
                    const int out = nt * 8 + g, in = kmap<MODE>(ks, h, t);
                    const bool ok = out < Cfg::n && in < Cfg::n;
                    const T v = ok ? sc.K[ok ? out : 0][ok ? in : 0] : (T)0;
                    if constexpr (MODE == MM_F64) {
                        hi[ks][nt][h] = v;
                    } else {
                        const uint32_t vh = to_tf32(v);
                        hi[ks][nt][h] = vh;
                        if constexpr (MODE == MM_TF32X3) lo[ks][nt][h] = to_tf32(v - tf32_value(vh));
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

// acc[mt] += K applied along the line whose 8-byte units at element kmap(ks, h, t) are ld(ks, h, u[MTW]) for the warp's m-tiles:
// a double (FP64, fragment row g) or a float2 = (fragment row g, fragment row g + 8) (TF32)
template <int P, int MODE, typename LD>
__device__ __forceinline__ void contract(Acc<P, MODE> (&acc)[MmaCfg<P, MODE>::MTW], const BFrags<P, MODE>& bf, int t, LD ld) {
    using Cfg = MmaCfg<P, MODE>;
    using T = typename Cfg::T;
    using U = typename std::conditional<MODE == MM_F64, double, float2>::type;
#pragma unroll
    for (int ks = 0; ks < Cfg::KS; ++ks) {
        constexpr int MTW = Cfg::MTW;
        T a[MTW][Cfg::NR][Cfg::KH];
#pragma unroll
        for (int h = 0; h < Cfg::KH; ++h) {
            // the last k-step is only partly populated: lanes beyond the line contribute zeros
            const bool all = kmap<MODE>(ks, h, 3) < Cfg::n;
            const bool ok = all || kmap<MODE>(ks, h, t) < Cfg::n;
            U u[MTW];
            if (ok) ld(ks, h, u);
#pragma unroll
            for (int mt = 0; mt < MTW; ++mt) {
                if constexpr (MODE == MM_F64) {
                    a[mt][0][h] = ok ? u[mt] : 0.0;
                } else {
                    a[mt][0][h] = ok ? u[mt].x : 0.f; a[mt][1][h] = ok ? u[mt].y : 0.f;
                }
            }
        }
#pragma unroll
        for (int mt = 0; mt < MTW; ++mt) {
            if constexpr (MODE == MM_F64) {
#pragma unroll
                for (int nt = 0; nt < Cfg::NT; ++nt) mma_f64(acc[mt].d[nt], a[mt][0][0], bf.hi[ks][nt][0]);
            } else {
                uint32_t ah[2][2], al[2][2];
#pragma unroll
                for (int r = 0; r < 2; ++r)
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        ah[r][h] = to_tf32(a[mt][r][h]);
                        if constexpr (MODE == MM_TF32X3) al[r][h] = to_tf32(a[mt][r][h] - tf32_value(ah[r][h]));
                    }
#pragma unroll
                for (int nt = 0; nt < Cfg::NT; ++nt) {
                    if constexpr (MODE == MM_TF32X3) {
                        mma_tf32(acc[mt].d[nt], al, bf.hi[ks][nt]);            // small terms first
                        mma_tf32(acc[mt].d[nt], ah, bf.lo[ks][nt]);
                    }
                    mma_tf32(acc[mt].d[nt], ah, bf.hi[ks][nt]);
                }
            }
        }
    }
}

template <int P, int MODE, bool HASPH, bool FULLV>
__global__ void __launch_bounds__(MmaCfg<P, MODE>::THREADS, 1)
cell_mma_kernel(const __grid_constant__ MmaConst<typename MmaCfg<P, MODE>::T> sc, const __grid_constant__ MarchArgs ar,
                const __grid_constant__ MarchMaps mp) {
    using Cfg = MmaCfg<P, MODE>;
    using T = typename Cfg::T;
    constexpr bool F64 = MODE == MM_F64;
    using U = typename std::conditional<F64, double, float2>::type;      // the thread's 8-byte unit of a node row
    constexpr int n = Cfg::n, C = Cfg::C, S = Cfg::S, RS = Cfg::RS, XPU = Cfg::XPU, NR = Cfg::NR, NT = Cfg::NT;
    constexpr int ESZ = Cfg::ESZ, KS = Cfg::KS, KH = Cfg::KH, MTW = Cfg::MTW;
    extern __shared__ unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full_in[S], empty_in[S], full_r[RS], empty_r[RS];
    // the swizzle is a function of shared-memory address bits: work from a 1024-byte aligned base
    unsigned char* const smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    U* const XRb = reinterpret_cast<U*>(smem + Cfg::XR_OFF);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int ROWB = (C / 2) * ESZ;
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
            int s = 0, rs = 0, ps = 0, prs = 0;               // ring slots and their phase parities
            for (int t = 0; t < T_; ++t) {
                mbar_wait(&empty_in[s], ps ^ 1);
                mbar_expect_tx(&full_in[s], Cfg::IN_BYTES);
                unsigned char* st = smem + (size_t)s * Cfg::IN_STAGE;
                int gz = g0 + t; if (gz == ar.n1[2]) gz = 0;
                const int line = gz * ar.n1[1] + ey * P;        // first x-line of the footprint in plane gz
                const int wline = gz * ar.n1[1];                // the y-wrapped line P of the last cell row
                const int xr = 2 * ex * P;                      // first (node, spin) row of the cell in its x-line
                if (!xwrap) {
                    // the face column x = P is the next node of every line: one box of 2(P+1) rows per line
                    if (!ywrap) {
                        tma_load_3d(st, &mp.main[0], col0, xr, line, &full_in[s]);
                    } else {
                        tma_load_3d(st, &mp.main[1], col0, xr, line, &full_in[s]);
                        tma_load_3d(st + P * Cfg::LINE_BYTES, &mp.main[2], col0, xr, wline, &full_in[s]);
                    }
                } else {
                    // last cell in x: node P of a line is the line's node 0 -- per line, 2P rows and then the 2 wrapped rows
                    for (int j = 0; j < n; ++j) {
                        const int gl = (j == P && ywrap) ? wline : line + j;
                        tma_load_3d(st + j * Cfg::LINE_BYTES, &mp.face[0], col0, xr, gl, &full_in[s]);
                        tma_load_3d(st + j * Cfg::LINE_BYTES + P * 128, &mp.face[1], col0, 0, gl, &full_in[s]);
                    }
                }
                if (t < T_ - 1) {                               // owned plane: R and the packed fields for S5
                    mbar_wait(&empty_r[rs], prs ^ 1);
                    mbar_expect_tx(&full_r[rs], Cfg::F_BYTES + (ar.useR ? Cfg::R_BYTES : 0));
                    unsigned char* rt = smem + Cfg::R_OFF + (size_t)rs * Cfg::R_STAGE;
                    if (ar.useR) tma_load_3d(rt, &mp.R, col0, xr, line, &full_r[rs]);
                    tma_load_2d_hint(rt + Cfg::R_BYTES, &mp.F, 4 * ex * P, line, &full_r[rs], pol_last);
                    if (++rs == RS) { rs = 0; prs ^= 1; }
                }
                if (++s == S) { s = 0; ps ^= 1; }
            }
        }
        return;
    }

    // ================================ consumers ================================
    // warp = index q in 0..p: row j of the X and Z tasks, x-position i of the Y task; it runs both m-tiles (mt = 0, 1: the two
    // halves of the CTA's vectors), whose units sit 32 bytes apart in a node row
    const int q = warp / (2 / MTW), mt0 = warp % (2 / MTW);
    const int g = lane >> 2, t4 = lane & 3;
    // the thread's 8-byte unit inside a node's 128-byte row: bit 3 = g & 1, spin (bit 6) = (g >> 1) & 1, chunk = 2 mt + (g >> 2)
    const int spin = (g >> 1) & 1;
    const uint32_t fb0 = (uint32_t)(spin * 64 + (2 * mt0 + (g >> 2)) * 16 + (g & 1) * 8);   // first m-tile of the warp; the next is 32 bytes on
    const int upos = (int)(fb0 >> 3);             // unit index inside the node (XR); m-tile 1: + 4
    // TF32: unit = complex64 of vector vl; FP64: unit = the re (ri = 0) or im (ri = 1) part of vector vl; m-tile 1: vl + VSTEP
    constexpr int VSTEP = F64 ? 2 : 4;
    const int vl = (F64 ? (g >> 2) : 2 * (g >> 2) + (g & 1)) + VSTEP * mt0;
    const int ri = F64 ? (g & 1) : 0;
    const double sgs = spin == 0 ? 1.0 : -1.0;    // sign of B_y in (B_x -+ i B_y)
    const int NTH = Cfg::NCW * 32;
    BFrags<P, MODE> bf;
    bf.init(sc, g, t4);
    const int v = chunk * Cfg::NV + vl;
    bool vok[MTW];
    double cin[MTW], cR[MTW];
#pragma unroll
    for (int mt = 0; mt < MTW; ++mt) {
        vok[mt] = FULLV || v + VSTEP * mt < ar.nvec;
        cin[mt] = (vok[mt] && ar.cin) ? __ldg(ar.cin + v + VSTEP * mt) : 0.0;
        cR[mt] = (vok[mt] && ar.cR && ar.useR) ? __ldg(ar.cR + v + VSTEP * mt) : 0.0;
    }
    constexpr int OSTEP = 2 * VSTEP;              // scalars of T between the two m-tiles' outputs
    // `out` offsets in scalars of T: node I -> 4 ld I; spin -> 2 ld; vector v -> 2 v (+ ri)
    const long long XS = 4 * ar.ld_out, LS = (long long)ar.n1[0] * XS, PS = (long long)ar.n1[1] * LS;
    const long long ocol0 = ((long long)spin * ar.ld_out + (vok[0] ? v : 0)) * 2 + ri;
    T* const outp = reinterpret_cast<T*>(ar.out);
    auto xoff = [&](int i) { int gx = ex * P + i; if (gx == ar.n1[0]) gx = 0; return (long long)gx * XS; };
    auto yoff = [&](int j) { int gy = ey * P + j; if (gy == ar.n1[1]) gy = 0; return (long long)gy * LS; };
    auto zoff = [&](int gzp) { if (gzp == ar.n1[2]) gzp = 0; return (long long)gzp * PS; };
    // this thread's output rows: 2 t4 + e of the first n-tile, and row 8 + 2 t4 + e of the second (live only where < n)
    const long long yq0 = yoff(2 * t4) + ocol0, yq1 = yoff(2 * t4 + 1 < n ? 2 * t4 + 1 : 0) + ocol0;
    const long long yq8 = yoff(8 + 2 * t4 < n ? 8 + 2 * t4 : 0) + ocol0, yq9 = yoff(9 + 2 * t4 < n ? 9 + 2 * t4 : 0) + ocol0;
    const long long xq_self = xoff(q);
    const long long zrow = yoff(q) + ocol0;
    const bool xph = HASPH && xwrap && ar.phd[0], yph = HASPH && ywrap && ar.phd[1];
    const T WXq = sc.W[0][q], WYq = sc.W[1][q];
    const T sXWY = sc.sdir[0] * WYq, sYWX = sc.sdir[1] * WXq;
    // fragment-load offsets inside a plane stage (bytes, before the swizzle)
    uint32_t xa[KS][KH], ya[KS][KH];
#pragma unroll
    for (int ks = 0; ks < KS; ++ks)
#pragma unroll
        for (int h = 0; h < KH; ++h) {
            const int kk = kmap<MODE>(ks, h, t4) < n ? kmap<MODE>(ks, h, t4) : 0;
            xa[ks][h] = (uint32_t)(q * n + kk) * 128u + fb0;
            ya[ks][h] = (uint32_t)(kk * n + q) * 128u + fb0;
        }
    auto ldu = [&](uint32_t lin) { return *reinterpret_cast<const U*>(smem + swz64(lin)); };
    // the units of both m-tiles at (m-tile 0) offset lin: bit 5 of lin is clear, so "+ 32" commutes with the swizzle as "^ 32"
    auto ldu2 = [&](uint32_t lin, U (&u)[MTW]) {
        const uint32_t a = swz64(lin);
        u[0] = *reinterpret_cast<const U*>(smem + a);
        if constexpr (MTW == 2) u[1] = *reinterpret_cast<const U*>(smem + (a ^ 32u));
    };

    // a complex output value held as d[0] = re, d[1] = im (TF32) or as the component ri of it (FP64, partner in lane ^ 4)
    struct Val { T a, b; };
    // multiply by conj(phase) = pr - i pi
    auto conj_phase = [&](Val x, double pr, double pi) {
        if constexpr (F64) {
            const double other = __shfl_xor_sync(0xffffffffu, x.a, 4);
            x.a = fma(other, ri ? -pi : pi, x.a * pr);                   // re' = re pr + im pi ; im' = im pr - re pi
        } else {
            const float re = (float)fma((double)x.b, pi, (double)x.a * pr), im = (float)fma((double)x.a, -pi, (double)x.b * pr);
            x.a = re; x.b = im;
        }
        return x;
    };
    auto emit = [&](T* p, Val x) {
        if constexpr (F64) red_add_t(p, x.a);
        else red_add_c64(p, x.a, x.b);
    };

    // ---- X task of plane tp (ring slot base sb, R slot rsl): x-contraction of row q and S5 on its owned nodes -> XR[tp & 1]
    auto xtask = [&](int tp, uint32_t sb, int rsl, int rpar, bool up, T inv_wz) {
        if (HASPH) {
            // Bloch phase on wrapped entries of the landed plane (x: node P of every line; y: line P; z: the whole wrapped
            // plane), fixed up in place before any task reads the plane (boundary CTAs only); this warp fixes row q
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
                    const uint32_t ea = swz64(sb + (uint32_t)(q * n + (valid ? i : 0)) * 128u + fb0);
#pragma unroll
                    for (int mt = 0; mt < MTW; ++mt) {
                        U* e = reinterpret_cast<U*>(smem + (ea ^ (mt ? 32u : 0u)));
                        if constexpr (F64) {
                            const double val = valid ? *e : 0.0;
                            const double other = __shfl_xor_sync(0xffffffffu, val, 4);
                            if (valid && (rowph || fx)) *e = fma(other, ri ? pi : -pi, val * pr);   // re' = re pr - im pi ; im' = im pr + re pi
                        } else {
                            if (valid && (rowph || fx)) {
                                const float2 z = *e;
                                *e = make_float2((float)fma((double)z.y, -pi, (double)z.x * pr), (float)fma((double)z.x, pi, (double)z.y * pr));
                            }
                        }
                    }
                }
                // these stage bytes are later rewritten by TMA.  No barrier here: this warp's X task reads only the units it
                // fixed; every other reader of the plane (Y and Z tasks) runs after the barrier that ends the step.
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
            }
        }
        Acc<P, MODE> acc[MTW];
#pragma unroll
        for (int mt = 0; mt < MTW; ++mt) acc[mt].zero();
        contract<P, MODE>(acc, bf, t4, [&](int ks, int h, U (&u)[MTW]) { ldu2(sb + xa[ks][h], u); });
        U* XR = XRb + (size_t)(tp & 1) * (Cfg::XR_BYTES / 8) + (q * n) * XPU + upos;
        const bool s5on = up && q < P;
        if (s5on) mbar_wait(&full_r[rsl], rpar);
        const uint32_t rb = Cfg::R_OFF + (uint32_t)rsl * Cfg::R_STAGE;
        const double* Fs = reinterpret_cast<const double*>(smem + rb + Cfg::R_BYTES) + (q * P) * 4;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                if (nt * 8 + e >= n) continue;                           // nothing in this fragment column at all
                const int xo = nt * 8 + 2 * t4 + e;
                const bool live = nt * 8 + 6 + e < n || xo < n;          // compile-time true for fully populated n-tiles
                const int xoc = live ? xo : 0;
                const bool own_node = s5on && live && (nt * 8 + 6 + e < P || xoc < P);
                Val val[MTW];
#pragma unroll
                for (int mt = 0; mt < MTW; ++mt) {
                    val[mt].a = sXWY * acc[mt].d[nt][0][e];
                    val[mt].b = NR == 2 ? sXWY * acc[mt].d[nt][NR - 1][e] : (T)0;
                }
                if (own_node) {
                    // S5 on an owned node: eq. 12 spin blocks, in-term, R-term, divided by the plane's
                    // z-weight because the Y task multiplies the whole XR entry by it
                    const double fd = Fs[xoc * 4 + spin], bx = Fs[xoc * 4 + 2], by = sgs * Fs[xoc * 4 + 3];
                    const uint32_t lin = sb + (uint32_t)(q * n + xoc) * 128u + fb0;
                    U me[MTW], ot[MTW];
                    ldu2(lin, me);
                    ldu2(lin ^ 64u, ot);
                    if constexpr (F64) {
                        // own component ri of spin s; the other spin's same (ot) and other (of) component
                        U of[MTW];
                        ldu2(lin ^ 72u, of);
                        const uint32_t rs0 = swz64(rb + (uint32_t)(q * P + xoc) * 128u + fb0);
#pragma unroll
                        for (int mt = 0; mt < MTW; ++mt) {
                            // s = 0: (B_x - i B_y) u' ; s = 1: (B_x + i B_y) u' ; re: B_x c + sgs B_y d ; im: B_x d - sgs B_y c
                            const double pot = fma(fd, me[mt], fma(bx, ot[mt], (ri ? -by : by) * of[mt]));
                            double s5 = fma(cin[mt], me[mt], sc.cHp * pot);
                            if (ar.useR) s5 = fma(cR[mt], *reinterpret_cast<const double*>(smem + (rs0 ^ (mt ? 32u : 0u))), s5);
                            val[mt].a = fma(s5, inv_wz, val[mt].a);
                        }
                    } else {
                        // R is complex128: the (node, spin) row is 16 doubles = 128 bytes, vector vl at byte 16 vl; m-tile 1 is
                        // 4 vectors = 64 bytes on (bit 6 of the offset is clear for m-tile 0)
                        const uint32_t rs0 = swz128(rb + (uint32_t)((q * P + xoc) * 2 + spin) * 128u + (uint32_t)vl * 16u);
                        // FP32 arithmetic ("pointwise terms stay FP32", A7); the R-term is formed in FP64 and rounded once
                        const float fdf = (float)fd, bxf = (float)bx, byf = (float)by, chp = (float)sc.cHp;
#pragma unroll
                        for (int mt = 0; mt < MTW; ++mt) {
                            const float a = me[mt].x, b = me[mt].y, c = ot[mt].x, d = ot[mt].y;
                            const float pre = fmaf(fdf, a, fmaf(bxf, c, byf * d)), pim = fmaf(fdf, b, fmaf(bxf, d, -byf * c));
                            float sre = fmaf((float)cin[mt], a, chp * pre), sim = fmaf((float)cin[mt], b, chp * pim);
                            if (ar.useR) {
                                const double2 rv = *reinterpret_cast<const double2*>(smem + (rs0 ^ (mt ? 64u : 0u)));
                                sre += (float)(cR[mt] * rv.x); sim += (float)(cR[mt] * rv.y);
                            }
                            val[mt].a = fmaf(sre, inv_wz, val[mt].a);
                            val[mt].b = fmaf(sim, inv_wz, val[mt].b);
                        }
                    }
                }
                if (live) {
#pragma unroll
                    for (int mt = 0; mt < MTW; ++mt) {
                        if constexpr (F64) XR[xoc * XPU + 4 * mt] = val[mt].a;
                        else XR[xoc * XPU + 4 * mt] = make_float2(val[mt].a, val[mt].b);
                    }
                }
            }
        if (up) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_r[rsl]);
        }
    };

    // ---- Y task of plane tp: y-contraction at x-position q, + XR (x part and S5), times the plane's z-weight -> RED to out
    auto ytask = [&](int tp, uint32_t sb, T wz) {
        Acc<P, MODE> acc[MTW];
#pragma unroll
        for (int mt = 0; mt < MTW; ++mt) acc[mt].zero();
        contract<P, MODE>(acc, bf, t4, [&](int ks, int h, U (&u)[MTW]) { ldu2(sb + ya[ks][h], u); });
        const U* XR = XRb + (size_t)(tp & 1) * (Cfg::XR_BYTES / 8) + q * XPU + upos;
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
        T* const pbase = outp + zoff(g0 + tp) + xq_self;
        auto outputs = [&](auto ph) {
            constexpr bool PH = decltype(ph)::value;
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    if (nt * 8 + e >= n) continue;
                    const int yo = nt * 8 + 2 * t4 + e;
                    const bool live = nt * 8 + 6 + e < n || yo < n;
                    const int yoc = live ? yo : 0;
                    const long long yq = nt == 0 ? (e == 0 ? yq0 : yq1) : (e == 0 ? yq8 : yq9);
#pragma unroll
                    for (int mt = 0; mt < MTW; ++mt) {
                        const U xr = XR[(yoc * n) * XPU + 4 * mt];
                        Val val;
                        if constexpr (F64) { val.a = wz * fma(sYWX, acc[mt].d[nt][0][e], xr); val.b = 0; }
                        else { val.a = wz * fmaf(sYWX, acc[mt].d[nt][0][e], xr.x); val.b = wz * fmaf(sYWX, acc[mt].d[nt][NR - 1][e], xr.y); }
                        if constexpr (PH) val = conj_phase(val, yoc == P ? pr1 : pr0, yoc == P ? pi1 : pi0);
                        if (live && vok[mt]) emit(pbase + yq + OSTEP * mt, val);
                    }
                }
        };
        // a real (warp-uniform) branch: the phase arithmetic must not be if-converted into the common path
        if (anyph) outputs(std::true_type{});
        else outputs(std::false_type{});
    };

    // ---- Z task of the cell whose planes sit in ring slots sl0, sl0+1, ... (mod S), first plane tb: z-contraction for the
    //      nodes of row q -> RED to out
    auto ztask = [&](int tb, int sl0) {
        uint32_t zb[KS][KH];                       // this lane's planes: stage base + the row's first node
#pragma unroll
        for (int ks = 0; ks < KS; ++ks)
#pragma unroll
            for (int h = 0; h < KH; ++h) {
                const int kk = kmap<MODE>(ks, h, t4) < n ? kmap<MODE>(ks, h, t4) : 0;
                int sl = sl0 + kk; if (sl >= S) sl -= S;
                zb[ks][h] = (uint32_t)sl * Cfg::IN_STAGE + (uint32_t)(q * n) * 128u + fb0;
            }
        const bool zwrap = (g0 + tb + P) == ar.n1[2];
        const bool zp = HASPH && zwrap && ar.phd[2];
        // this thread's output planes: tb + 2 t4 + e, and tb + 8 + 2 t4 + e (live only where < n)
        const long long zq0 = zoff(g0 + tb + 2 * t4) + zrow, zq1 = zoff(g0 + tb + (2 * t4 + 1 < n ? 2 * t4 + 1 : 0)) + zrow;
        const long long zq8 = zoff(g0 + tb + (8 + 2 * t4 < n ? 8 + 2 * t4 : 0)) + zrow;
        const long long zq9 = zoff(g0 + tb + (9 + 2 * t4 < n ? 9 + 2 * t4 : 0)) + zrow;
#pragma unroll 1
        for (int i = 0; i < n; ++i) {                 // (unrolling by 3 to put three nodes in flight changed nothing: 6.42 vs 6.37 ms)
            Acc<P, MODE> acc[MTW];
#pragma unroll
            for (int mt = 0; mt < MTW; ++mt) acc[mt].zero();
            const uint32_t no = (uint32_t)i * 128u;
            contract<P, MODE>(acc, bf, t4, [&](int ks, int h, U (&u)[MTW]) { ldu2(zb[ks][h] + no, u); });
            const T w = sc.W[0][i] * WYq;
            const bool anyph = HASPH && ((i == P && xph) || (q == P && yph) || zp);
            double pr0 = 1.0, pi0 = 0.0, pr1 = 1.0, pi1 = 0.0;          // conj phase of planes < P / of the wrapped top plane
            if (anyph) {
                if (i == P && xph) { pr0 = ar.ph_re[0]; pi0 = ar.ph_im[0]; }
                if (q == P && yph) { const double u = pr0 * ar.ph_re[1] - pi0 * ar.ph_im[1]; pi0 = pr0 * ar.ph_im[1] + pi0 * ar.ph_re[1]; pr0 = u; }
                pr1 = pr0; pi1 = pi0;
                if (zp) { pr1 = pr0 * ar.ph_re[2] - pi0 * ar.ph_im[2]; pi1 = pr0 * ar.ph_im[2] + pi0 * ar.ph_re[2]; }
            }
            T* const nb = outp + xoff(i);
            auto outputs = [&](auto ph) {
                constexpr bool PH = decltype(ph)::value;
#pragma unroll
                for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        if (nt * 8 + e >= n) continue;
                        const int ko = nt * 8 + 2 * t4 + e;
                        const bool live = nt * 8 + 6 + e < n || ko < n;
                        const int koc = live ? ko : 0;
                        const long long zq = nt == 0 ? (e == 0 ? zq0 : zq1) : (e == 0 ? zq8 : zq9);
#pragma unroll
                        for (int mt = 0; mt < MTW; ++mt) {
                            Val val;
                            val.a = w * acc[mt].d[nt][0][e];
                            val.b = NR == 2 ? w * acc[mt].d[nt][NR - 1][e] : (T)0;
                            if constexpr (PH) val = conj_phase(val, koc == P ? pr1 : pr0, koc == P ? pi1 : pi0);
                            if (live && vok[mt]) emit(nb + zq + OSTEP * mt, val);
                        }
                    }
            };
            if (anyph) outputs(std::true_type{});
            else outputs(std::false_type{});
        }
    };

    // ---- march.  Plane t sits in ring slot t mod S (sl), its R / fields in slot t mod RS; c = t mod P is its index in the
    //      cell above it.  In-plane weight of plane t: W_z[c] for the cell above (if any) + W_z[P] for the cell below (if any).
    auto zweight = [&](int t, int c) {
        return (t < T_ - 1 ? sc.W[2][c] : (T)0) + ((c == 0 && t > 0) ? sc.W[2][P] : (T)0);
    };
    mbar_wait(&full_in[0], 0);
    xtask(0, 0u, 0, 0, true, (T)1 / zweight(0, 0));
    asm volatile("bar.sync 1, %0;" ::"r"(NTH) : "memory");
    int c = 0, sl = 0, par = 0;                    // of plane t
    int rsl = 1 % RS, rpar = (1 / RS) & 1;         // R slot / parity of plane t + 1
    int cell_sl = 0;                               // ring slot of the first plane of the cell being filled
#pragma unroll 1
    for (int t = 0; t < T_; ++t) {
        const bool lower = c == 0 && t > 0, upper = t < T_ - 1;
        int sl1 = sl + 1, par1 = par; if (sl1 == S) { sl1 = 0; par1 ^= 1; }
        const int c1 = (c + 1 == P) ? 0 : c + 1;
        if (upper) {
            mbar_wait(&full_in[sl1], par1);
            // XR[(t+1)&1] was last read in the Y task of plane t-1, before the last barrier
            xtask(t + 1, (uint32_t)sl1 * Cfg::IN_STAGE, rsl, rpar, t + 1 < T_ - 1, (T)1 / zweight(t + 1, c1));
            if (++rsl == RS) { rsl = 0; rpar ^= 1; }
        }
        ytask(t, (uint32_t)sl * Cfg::IN_STAGE, zweight(t, c));
        if (lower) {
            ztask(t - P, cell_sl);                 // the cell below is complete and all its planes are still resident
            __syncwarp();
            if (lane == 0) {
                int k = cell_sl;
                for (int j = 0; j < P; ++j) { mbar_arrive(&empty_in[k]); if (++k == S) k = 0; }   // its planes but the shared top one
            }
            cell_sl = sl;
        }
        asm volatile("bar.sync 1, %0;" ::"r"(NTH) : "memory");
        c = c1; sl = sl1; par = par1;
    }
}

// ---------------------------------------------------------------------------------------------
// All scalings (1/2, Jacobian, D^-1 on the way in, M^-1 on the way out, the step coefficient) folded into the 1-D tables.
// On this mesh the three scaled 1-D operators are one matrix times a scalar per direction (the directions differ only in
// h_d): the kernel keeps the z-direction matrix and the two ratios.
template <typename T>
static bool build_mma_const(const chfsi_mesh* m, const CellArgs& a, MmaConst<T>& sc) {
    const MeshConst& mc = m->mc;
    const int n = mc.n;
    const bool sin_ = (a.flags & kScaleIn) != 0, sout_ = (a.flags & kSoutInvM) != 0;
    std::memset(&sc, 0, sizeof(sc));
    sc.cHp = a.cH;
    double K[3][kMaxN][kMaxN];
    for (int d = 0; d < 3; ++d)
        for (int i = 0; i < n; ++i) {
            const double si = sin_ ? mc.im1[d][i] : 1.0, so = sout_ ? mc.im1[d][i] : 1.0;
            for (int b = 0; b < n; ++b) {
                const double sb = sin_ ? mc.im1[d][b] : 1.0;
                // the step coefficient rides on the x-direction factors: on K_x for the x part and on W_x for the y and z parts
                K[d][i][b] = (d == 0 ? a.cH : 1.0) * so * mc.Kd[d][i][b] * sb;
            }
            sc.W[d][i] = (T)((d == 0 ? a.cH : 1.0) * mc.w[i] * so * si);
        }
    if (K[2][0][0] == 0.0) return false;
    double amax = 0.0;
    for (int i = 0; i < n; ++i)
        for (int b = 0; b < n; ++b) { sc.K[i][b] = (T)K[2][i][b]; amax = std::fmax(amax, std::fabs(K[2][i][b])); }
    for (int d = 0; d < 3; ++d) {
        const double s = K[d][0][0] / K[2][0][0];
        for (int i = 0; i < n; ++i)
            for (int b = 0; b < n; ++b)
                if (std::fabs(K[d][i][b] - s * K[2][i][b]) > 1e-12 * std::fabs(s) * amax) return false;   // not proportional
        sc.sdir[d] = (T)s;
    }
    return true;
}

static std::once_flag g_mma_attr_once[4][3][4][32];   // [p/2 - 1][mode][phase, full tiles][device]

template <int P, int MODE>
static cudaError_t launch_mma_t(const chfsi_mesh* m, const CellArgs& a, cudaStream_t st) {
    using Cfg = MmaCfg<P, MODE>;
    using T = typename Cfg::T;
    MmaConst<T> sc;
    if (!build_mma_const<T>(m, a, sc)) return cudaErrorInvalidValue;
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
    const int sw64 = kSwizzle ? 64 : 0, sw128 = kSwizzle ? 128 : 0;
    // with a single cell in x the 2(P+1)-row box would not fit the x-line: such meshes always take the per-line path
    const int rows_full = ar.nc[0] > 1 ? 2 * (P + 1) : 2 * P;
    for (int i = 0; i < 3; ++i)
        if (!make_map3(&mp.main[i], m, a.in, a.ld_in, a.nvec, BC, rows_full, nl[i], f32, sw64)) return cudaErrorInvalidValue;
    if (!make_map3(&mp.face[0], m, a.in, a.ld_in, a.nvec, BC, 2 * P, 1, f32, sw64) ||
        !make_map3(&mp.face[1], m, a.in, a.ld_in, a.nvec, BC, 2, 1, f32, sw64) ||
        !make_map3(&mp.face[2], m, a.in, a.ld_in, a.nvec, BC, 2, 1, f32, sw64))
        return cudaErrorInvalidValue;
    // R is complex128 in every mode: its (node, spin) row is 128 bytes with complex64 iterates, 64 bytes with complex128 ones
    if (!make_map3(&mp.R, m, ar.useR ? a.R : a.in, ar.useR ? a.ld_R : a.ld_in, a.nvec, BC, 2 * P, P, ar.useR ? false : f32,
                   f32 ? sw128 : sw64) ||
        !make_mapF(&mp.F, m, P))
        return cudaErrorInvalidValue;
    if (a.flags & kMassIn) return cudaErrorInvalidValue;             // the residual S0 runs on the line-owned FP64 kernel
    const bool ph = m->mc.has_phase != 0, full = a.nvec % Cfg::NV == 0;
    auto kern = ph ? (full ? cell_mma_kernel<P, MODE, true, true> : cell_mma_kernel<P, MODE, true, false>)
                   : (full ? cell_mma_kernel<P, MODE, false, true> : cell_mma_kernel<P, MODE, false, false>);
    cudaError_t attr_err = cudaSuccess;
    std::call_once(g_mma_attr_once[P / 2 - 1][MODE][(ph ? 2 : 0) + (full ? 1 : 0)][m->device & 31], [&] {
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
