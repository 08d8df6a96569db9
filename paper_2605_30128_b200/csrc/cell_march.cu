// Z-marching cell kernel (FP64): the dominant kernel of the filter on sm_100a.
//
// One CTA owns the xy-footprint of one FE cell column (ex, ey), a z-segment of `cps` cells and NV = 8
// complex vectors (C = 32 real batch columns = one warp wide), and marches through the xy-planes of
// that column:
//   producer warp : one elected thread streams each plane -- (p+1)^2 gathered node rows of `in`, the
//                   p^2 owned rows of R and the packed local fields -- into a ring of shared-memory
//                   stages with TMA (cp.async.bulk.tensor.2d, one box per y-line; the periodic wrap in
//                   x is a second 2-row box) completing on an mbarrier (S1 gather, PAPER.md:204 (i)).
//   consumer warps: warp j owns y-row j of the footprint, lane = batch column.  Per plane it does the
//                   x-contraction on its own row in registers, the y-contraction by reading the plane's
//                   columns, and *pushes* the plane into the (p+1) z-accumulators of the current cell
//                   (S2: three 1-D contractions; the z one never touches memory).
//                   The 2x2 spin potential (eq. 12), the in-term and the R-term of eq. 11 (S5) are added
//                   to the accumulator of the node's own plane.  When a cell is finished its p planes are
//                   emitted with one RED.ADD.F64 per node and column (S3, PAPER.md:204 (iii)); the top plane
//                   carries over to the next cell, so z-faces are assembled in registers.
// All scalings (1/2, Jacobian, D^-1 on the way in, M^-1 on the way out, the step coefficient) are folded
// into the per-launch 1-D tables (StepConst), so the inner loops are bare FMAs with immediate operands.
#include <cuda.h>

#include <cstring>
#include <type_traits>

#include "chfsi_internal.h"

namespace chfsi {

struct StepConst {
    double KX[kMaxN][kMaxN];   // cH * sout_x[i] * Kx[i][a] * sin_x[a]
    double KY[kMaxN][kMaxN];
    double KZ[kMaxN][kMaxN];
    double WX[kMaxN], WY[kMaxN], WZ[kMaxN];   // w * sout * sin per direction
    double PX[kMaxN], PY[kMaxN], PZ[kMaxN];   // product = cH * s_out * (u/in)   (potential coefficient)
    double FX[kMaxN], FY[kMaxN], FZ[kMaxN];   // product = in-term mass factor
};

struct MarchArgs {
    int nc[3], n1[3];
    int has_phase;
    double ph_re[3], ph_im[3];
    int nseg, cps;              // z segments, cells per segment
    int nvec, nchunks;
    int useR;
    const double* fields;       // [M][4] = V+Bz, V-Bz, Bx, By
    const double* cin;          // [nvec]
    const double* cR;           // [nvec] or null
    double* out;
    long long ld_out;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
    uint32_t ok = 0;
    const uint32_t a = smem_u32(b);
    while (!ok) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

template <int P>
struct MarchCfg {
    static constexpr int n = P + 1;
    static constexpr int C = 32;                          // real batch columns per CTA (NV = 8 complex)
    static constexpr int IN_BYTES = n * n * C * 8;
    static constexpr int R_BYTES = P * P * C * 8;
    static constexpr int F_BYTES = P * P * 32;
    static constexpr int R_OFF = IN_BYTES;
    static constexpr int F_OFF = IN_BYTES + R_BYTES;
    static constexpr int STAGE_BYTES = ((F_OFF + F_BYTES + 127) / 128) * 128;
    static constexpr int STAGES = (200 * 1024 / STAGE_BYTES) < 8 ? (200 * 1024 / STAGE_BYTES) : 8;
    static constexpr int THREADS = (n + 1) * 32;
};

// Per-thread state of a consumer warp (row j of the footprint, lane = batch column).
template <int P, bool HASPH>
struct MarchConsumer {
    using Cfg = MarchCfg<P>;
    static constexpr int n = Cfg::n, C = Cfg::C, STAGES = Cfg::STAGES;
    double acc[n][n];            // z-accumulators of the current cell: acc[k][a], plane k, x-position a
    double kyrow[n], wxy[n];
    double wyj, pyj, fyj, cin, cR;
    double* outcol;
    int j, col, s_spin, ri, ex, gy, g0;
    bool vok, jown, wy, xwrap, ywrap;

    __device__ __forceinline__ void init(const StepConst& sc, const MarchArgs& ar, int warp, int lane, int ex_, int ey,
                                         int chunk, int g0_, bool xw, bool yw) {
        j = warp; col = lane; ex = ex_; g0 = g0_; xwrap = xw; ywrap = yw;
        s_spin = col >> 4; ri = col & 1;
        const int vl = (col & 15) >> 1;
        const int v = chunk * 8 + vl;
        vok = v < ar.nvec;
        jown = j < P;
#pragma unroll
        for (int b = 0; b < n; ++b) { kyrow[b] = sc.KY[j][b]; wxy[b] = sc.WX[b] * sc.WY[j]; }
        wyj = sc.WY[j]; pyj = sc.PY[j]; fyj = sc.FY[j];
        cin = (vok && ar.cin) ? __ldg(ar.cin + v) : 0.0;
        cR = (vok && ar.cR && ar.useR) ? __ldg(ar.cR + v) : 0.0;
        gy = ey * P + j; wy = gy == ar.n1[1]; if (wy) gy = 0;
        outcol = ar.out + ((long long)s_spin * ar.ld_out + v) * 2 + ri;
#pragma unroll
        for (int k = 0; k < n; ++k)
#pragma unroll
            for (int a = 0; a < n; ++a) acc[k][a] = 0.0;
    }

    __device__ __forceinline__ static void phase_of(const MarchArgs& ar, bool wx, bool wyy, bool wz, double& pr, double& pi) {
        pr = 1.0; pi = 0.0;
        if (wx) { pr = ar.ph_re[0]; pi = ar.ph_im[0]; }
        if (wyy) { const double tt = pr * ar.ph_re[1] - pi * ar.ph_im[1]; pi = pr * ar.ph_im[1] + pi * ar.ph_re[1]; pr = tt; }
        if (wz) { const double tt = pr * ar.ph_re[2] - pi * ar.ph_im[2]; pi = pr * ar.ph_im[2] + pi * ar.ph_re[2]; pr = tt; }
    }

    // emit planes [0, nk) of the accumulators to global planes gzbase + k  (S3: one RED.ADD.F64 per node and column)
    __device__ __forceinline__ void emit(const MarchArgs& ar, int gzbase, int nk) {
        const long long xstride = 4 * ar.ld_out;                       // doubles between consecutive nodes
        const long long x0 = (long long)ex * P;
#pragma unroll
        for (int k = 0; k < n; ++k) {
            if (k < nk) {
                int gz = gzbase + k; const bool wz = gz == ar.n1[2]; if (wz) gz = 0;
                double* line = outcol + ((long long)gz * ar.n1[1] + gy) * ar.n1[0] * xstride;
                double* pnode = line + x0 * xstride;
#pragma unroll
                for (int a = 0; a < n; ++a) {
                    const bool wx = (a == P) && xwrap;
                    double* dst = wx ? line : pnode + a * xstride;
                    double val = acc[k][a];
                    if (HASPH) {
                        const double other = __shfl_xor_sync(0xffffffffu, val, 1);
                        if (wx | wy | wz) {
                            double pr, pi; phase_of(ar, wx, wy, wz, pr, pi);
                            val = ri == 0 ? val * pr + other * pi : val * pr - other * pi;   // times conj(phase)
                        }
                    }
                    if (vok) atomicAdd(dst, val);
                }
            }
        }
    }

    // One plane t of the march.  c = its local index in the current cell (upper role); lower: it is also plane P of
    // the previous cell; upper: it belongs to a cell of this segment (false only for the segment's last plane).
    __device__ __forceinline__ void plane(const StepConst& sc, const MarchArgs& ar, unsigned char* smem, uint64_t* full_bar,
                                          uint64_t* empty_bar, int t, int c, bool lower, bool upper) {
        const int s = t % STAGES;
        const uint32_t par = (t / STAGES) & 1;
        mbar_wait(&full_bar[s], par);
        double* IN = reinterpret_cast<double*>(smem + (size_t)s * Cfg::STAGE_BYTES);
        const double* Rs = reinterpret_cast<const double*>(smem + (size_t)s * Cfg::STAGE_BYTES + Cfg::R_OFF);
        const double* Fs = reinterpret_cast<const double*>(smem + (size_t)s * Cfg::STAGE_BYTES + Cfg::F_OFF);
        if (HASPH) {
            // Bloch phase on wrapped entries (x: column a = P; y: row j = P; z: the wrapped plane), fixed up in place
            const bool wz = (g0 + t) == ar.n1[2];
            if (xwrap | ywrap | wz) {
                const bool wyy = ywrap && j == P;
#pragma unroll 1
                for (int a = 0; a < n; ++a) {
                    const bool wx = xwrap && a == P;
                    if (wx | wyy | wz) {
                        double pr, pi; phase_of(ar, wx, wyy, wz, pr, pi);
                        const double val = IN[(j * n + a) * C + col];
                        const double other = __shfl_xor_sync(0xffffffffu, val, 1);
                        IN[(j * n + a) * C + col] = ri == 0 ? val * pr - other * pi : other * pi + val * pr;
                    }
                }
                asm volatile("bar.sync 1, %0;" ::"r"(n * 32) : "memory");   // consumer warps only
            }
        }
        const double* INc = IN + col;
        double row[n];
#pragma unroll
        for (int a = 0; a < n; ++a) row[a] = INc[(j * n + a) * C];
        double ip[n];
        // y-contraction: column a of the plane against row j of KY
#pragma unroll
        for (int a = 0; a < n; ++a) {
            double sy = 0.0;
#pragma unroll
            for (int b = 0; b < n; ++b) sy = fma(kyrow[b], INc[(b * n + a) * C], sy);
            ip[a] = sc.WX[a] * sy;
        }
        // x-contraction on the own row
#pragma unroll
        for (int i = 0; i < n; ++i) {
            double sx = 0.0;
#pragma unroll
            for (int a = 0; a < n; ++a) sx = fma(sc.KX[i][a], row[a], sx);
            ip[i] = fma(wyj, sx, ip[i]);
        }
        double zr[n];
#pragma unroll
        for (int a = 0; a < n; ++a) zr[a] = wxy[a] * row[a];
        if (lower) {
#pragma unroll
            for (int k = 0; k < n; ++k)
#pragma unroll
                for (int a = 0; a < n; ++a) acc[k][a] = fma(sc.KZ[k][P], zr[a], acc[k][a]);
#pragma unroll
            for (int a = 0; a < n; ++a) acc[P][a] = fma(sc.WZ[P], ip[a], acc[P][a]);
            // the previous cell is complete: emit its planes 0..P-1, carry its top plane over
            emit(ar, g0 + t - P, P);
#pragma unroll
            for (int a = 0; a < n; ++a) acc[0][a] = acc[P][a];
#pragma unroll
            for (int k = 1; k < n; ++k)
#pragma unroll
                for (int a = 0; a < n; ++a) acc[k][a] = 0.0;
        }
        if (upper) {
            // z-push with the runtime cell-local index c: column c of KZ fetched from the constant bank
#pragma unroll
            for (int k = 0; k < n; ++k) {
                const double kz = sc.KZ[k][c];
#pragma unroll
                for (int a = 0; a < n; ++a) acc[k][a] = fma(kz, zr[a], acc[k][a]);
            }
            const double wzc = sc.WZ[c];
#pragma unroll
            for (int a = 0; a < n; ++a) ip[a] *= wzc;
            if (jown) {
                // S5 on the owned nodes of this plane (a < P): eq. 12 spin blocks, in-term, R-term
                const double pz = sc.PZ[c] * pyj, fz = sc.FZ[c] * fyj * cin;
#pragma unroll
                for (int a = 0; a < P; ++a) {
                    const double in_own = row[a];
                    const double o_same = INc[(j * n + a) * C + ((col ^ 16) - col)];
                    const double o_flip = INc[(j * n + a) * C + ((col ^ 17) - col)];
                    const double u_re = ri == 0 ? o_same : o_flip;       // other spin, same vector
                    const double u_im = ri == 0 ? o_flip : o_same;
                    const double4 f = *reinterpret_cast<const double4*>(Fs + (j * P + a) * 4);
                    const double diag = s_spin == 0 ? f.x : f.y;
                    const double sy = s_spin == 0 ? -f.w : f.w;
                    const double offd = ri == 0 ? f.z * u_re - sy * u_im : f.z * u_im + sy * u_re;
                    double val = fma(pz * sc.PX[a], fma(diag, in_own, offd), ip[a]);
                    val = fma(fz * sc.FX[a], in_own, val);
                    if (ar.useR) val = fma(cR, Rs[(j * P + a) * C + col], val);
                    ip[a] = val;
                }
            }
            // add the in-plane + pointwise part to the accumulator of the plane's own index
#pragma unroll
            for (int k = 0; k < P; ++k) {
                if (c == k) {
#pragma unroll
                    for (int a = 0; a < n; ++a) acc[k][a] += ip[a];
                }
            }
        }
        __syncwarp();
        if (col == 0) mbar_arrive(&empty_bar[s]);
    }
};

template <int P, bool HASPH>
__global__ void __launch_bounds__(MarchCfg<P>::THREADS, 1)
cell_march_kernel(const __grid_constant__ StepConst sc, const __grid_constant__ MarchArgs ar,
                  const __grid_constant__ CUtensorMap map_in_full, const __grid_constant__ CUtensorMap map_in_p,
                  const __grid_constant__ CUtensorMap map_in_1, const __grid_constant__ CUtensorMap map_R) {
    using Cfg = MarchCfg<P>;
    constexpr int n = Cfg::n, C = Cfg::C, STAGES = Cfg::STAGES;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full_bar[STAGES], empty_bar[STAGES];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // blockIdx -> (ex fastest, ey, seg, chunk): neighbours in x/y run together, so shared faces hit in L2
    int bid = blockIdx.x;
    const int ex = bid % ar.nc[0]; bid /= ar.nc[0];
    const int ey = bid % ar.nc[1]; bid /= ar.nc[1];
    const int seg = bid % ar.nseg;
    const int chunk = bid / ar.nseg;
    const int T = ar.cps * P + 1;                 // planes this CTA marches through
    const int g0 = seg * ar.cps * P;              // first global plane
    const bool xwrap = ex == ar.nc[0] - 1, ywrap = ey == ar.nc[1] - 1;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], n); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == n) {
        // ================================ producer ================================
        if (lane == 0) {
            const int col0 = chunk * 16;                          // doubles
            for (int t = 0; t < T; ++t) {
                const int s = t % STAGES;
                const uint32_t par = (t / STAGES) & 1;
                mbar_wait(&empty_bar[s], par ^ 1);
                const bool owned = t < T - 1;
                uint32_t bytes = Cfg::IN_BYTES;
                if (owned) bytes += Cfg::F_BYTES + (ar.useR ? Cfg::R_BYTES : 0);
                mbar_expect_tx(&full_bar[s], bytes);
                unsigned char* st = smem + (size_t)s * Cfg::STAGE_BYTES;
                int gz = g0 + t; if (gz == ar.n1[2]) gz = 0;
                for (int jj = 0; jj < n; ++jj) {
                    int gy = ey * P + jj; if (gy == ar.n1[1]) gy = 0;
                    const long long line0 = ((long long)gz * ar.n1[1] + gy) * ar.n1[0];   // node index of x = 0
                    const long long node0 = line0 + (long long)ex * P;
                    unsigned char* dst = st + jj * n * C * 8;
                    if (!xwrap) {
                        tma_load_2d(dst, &map_in_full, col0, (int)(2 * node0), &full_bar[s]);
                    } else {
                        tma_load_2d(dst, &map_in_p, col0, (int)(2 * node0), &full_bar[s]);
                        tma_load_2d(dst + P * C * 8, &map_in_1, col0, (int)(2 * line0), &full_bar[s]);
                    }
                    if (owned && jj < P) {
                        if (ar.useR) tma_load_2d(st + Cfg::R_OFF + jj * P * C * 8, &map_R, col0, (int)(2 * node0), &full_bar[s]);
                        bulk_load(st + Cfg::F_OFF + jj * P * 32, ar.fields + node0 * 4, P * 32, &full_bar[s]);
                    }
                }
            }
        }
        return;
    }

    // ================================ consumers ================================
    MarchConsumer<P, HASPH> cs;
    cs.init(sc, ar, warp, lane, ex, ey, chunk, g0, xwrap, ywrap);
    int c = 0;
#pragma unroll 1
    for (int t = 0; t < T; ++t) {
        cs.plane(sc, ar, smem, full_bar, empty_bar, t, c, c == 0 && t > 0, t < T - 1);
        c = (c + 1 == P) ? 0 : c + 1;
    }
    cs.emit(ar, g0 + T - 1, 1);                                   // partial of the segment's top face
}

// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                             const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeFn get_encode() {
    static EncodeFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeFn>(p);
    }
    return fn;
}

// 2-D view of a multivector: dim0 = 2*ld doubles of one (node, spin) row, dim1 = 2*M rows; box = 16 doubles x rows
static bool make_map(CUtensorMap* map, const double* base, long long ld, long long nrows, int box_rows) {
    EncodeFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t gdim[2] = {(cuuint64_t)(2 * ld), (cuuint64_t)nrows};
    cuuint64_t gstr[1] = {(cuuint64_t)(ld * 16)};
    cuuint32_t box[2] = {16u, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1u, 1u};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), gdim, gstr, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool march_supported(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a) {
    if (prec != CHFSI_FP64) return false;
    if (m->p != 2 && m->p != 4 && m->p != 6) return false;
    if (m->dF == nullptr) return false;
    // TMA needs 16-byte aligned bases/strides (always true for complex128 rows) and 32-bit row coordinates
    if (2 * m->nnodes >= (1ll << 31)) return false;
    if (((uintptr_t)a.in & 15) || ((uintptr_t)a.out & 15) || (a.R && ((uintptr_t)a.R & 15))) return false;
    return get_encode() != nullptr;
}

static void build_step_const(const chfsi_mesh* m, const CellArgs& a, StepConst& sc) {
    const MeshConst& mc = m->mc;
    const int n = mc.n;
    const bool sin_ = (a.flags & kScaleIn) != 0, sout_ = (a.flags & kSoutInvM) != 0, massin = (a.flags & kMassIn) != 0;
    std::memset(&sc, 0, sizeof(sc));
    for (int d = 0; d < 3; ++d) {
        double (*K)[kMaxN] = d == 0 ? sc.KX : d == 1 ? sc.KY : sc.KZ;
        double* W = d == 0 ? sc.WX : d == 1 ? sc.WY : sc.WZ;
        double* Pp = d == 0 ? sc.PX : d == 1 ? sc.PY : sc.PZ;
        double* Fp = d == 0 ? sc.FX : d == 1 ? sc.FY : sc.FZ;
        for (int i = 0; i < n; ++i) {
            const double si = sin_ ? mc.im1[d][i] : 1.0, so = sout_ ? mc.im1[d][i] : 1.0;
            for (int b = 0; b < n; ++b) {
                const double sb = sin_ ? mc.im1[d][b] : 1.0;
                K[i][b] = a.cH * so * mc.Kd[d][i][b] * sb;
            }
            W[i] = mc.w[i] * so * si;
            const double fu = sin_ ? 1.0 : mc.m1[d][i];                // u = m w: Z-form u = in, else m * in
            Pp[i] = so * fu * (d == 0 ? a.cH : 1.0);
            Fp[i] = massin ? mc.m1[d][i] : 1.0;
        }
    }
}

template <int P>
static cudaError_t launch_march_t(const chfsi_mesh* m, const CellArgs& a, cudaStream_t st) {
    using Cfg = MarchCfg<P>;
    StepConst sc;
    build_step_const(m, a, sc);
    MarchArgs ar;
    std::memset(&ar, 0, sizeof(ar));
    for (int d = 0; d < 3; ++d) {
        ar.nc[d] = m->mc.nc[d]; ar.n1[d] = m->mc.n1[d];
        ar.ph_re[d] = m->mc.ph_re[d]; ar.ph_im[d] = m->mc.ph_im[d];
    }
    ar.has_phase = m->mc.has_phase;
    ar.nvec = a.nvec; ar.nchunks = (a.nvec + 7) / 8;
    ar.useR = (a.R != nullptr && a.cR != nullptr) ? 1 : 0;
    ar.fields = m->dF; ar.cin = a.cin; ar.cR = a.cR; ar.out = a.out; ar.ld_out = a.ld_out;
    // z segmentation: enough CTAs for >= ~4 waves of one CTA per SM
    const long long base = (long long)ar.nc[0] * ar.nc[1] * ar.nchunks;
    int nseg = 1;
    for (int cand = 1; cand <= ar.nc[2]; ++cand)
        if (ar.nc[2] % cand == 0) { nseg = cand; if (base * cand >= 4 * 148) break; }
    ar.nseg = nseg; ar.cps = ar.nc[2] / nseg;
    CUtensorMap mf, mp, m1, mr;
    const long long rows = 2 * m->nnodes;
    if (!make_map(&mf, a.in, a.ld_in, rows, 2 * (P + 1)) || !make_map(&mp, a.in, a.ld_in, rows, 2 * P) ||
        !make_map(&m1, a.in, a.ld_in, rows, 2) ||
        !make_map(&mr, ar.useR ? a.R : a.in, ar.useR ? a.ld_R : a.ld_in, rows, 2 * P))
        return cudaErrorInvalidValue;
    const size_t smem = (size_t)Cfg::STAGES * Cfg::STAGE_BYTES;
    static bool attr_done[128] = {false};
    auto kern = m->mc.has_phase ? cell_march_kernel<P, true> : cell_march_kernel<P, false>;
    const int slot = (m->device & 63) * 2 + (m->mc.has_phase ? 1 : 0);
    if (!attr_done[slot]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_done[slot] = true;
    }
    const long long grid = base * nseg;
    kern<<<(unsigned)grid, Cfg::THREADS, smem, st>>>(sc, ar, mf, mp, m1, mr);
    return cudaGetLastError();
}

cudaError_t launch_cell_march(const chfsi_mesh* m, const CellArgs& a, cudaStream_t st) {
    switch (m->p) {
        case 2: return launch_march_t<2>(m, a, st);
        case 4: return launch_march_t<4>(m, a, st);
        case 6: return launch_march_t<6>(m, a, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace chfsi
