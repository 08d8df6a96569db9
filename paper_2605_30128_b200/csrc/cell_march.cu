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
#include "tma_util.cuh"

namespace chfsi {

struct StepConst {
    double KX[kMaxN][kMaxN];   // cH * sout_x[i] * Kx[i][a] * sin_x[a]
    double KY[kMaxN][kMaxN];
    double KZ[kMaxN][kMaxN];
    double WX[kMaxN], WY[kMaxN], WZ[kMaxN];   // w * sout * sin per direction
    double PX[kMaxN], PY[kMaxN], PZ[kMaxN];   // product = cH * s_out * (u/in)   (potential coefficient)
    double FX[kMaxN], FY[kMaxN], FZ[kMaxN];   // product = in-term mass factor
    // FP32 product (CHFSI_FP32): the same tables without cH, rounded once to FP32; cH is applied in FP64 when the
    // FP32 Laplacian is widened
    float KXf[kMaxN][kMaxN], KYf[kMaxN][kMaxN], KZf[kMaxN][kMaxN];
    float WXf[kMaxN], WYf[kMaxN], WZf[kMaxN];
    double cH;                 // FP32 product: step coefficient / in_scale, applied in FP64 to the widened Laplacian
    double in_scale;           // FP32 product: power of two applied (in FP64) to `in` before the cast
};

// Thread mapping of the consumers.  A consumer thread is (x-part h, footprint row j, batch column col):
//   warp w -> h = w / WPH;  j = (w % WPH) * RPW + lane / C;  col = lane % C.
// Part h owns the x-positions [h*NA, min(n, (h+1)*NA)) of its row: it computes the x-, y- and z-contractions
// only for those outputs, so the (p+1) z-accumulator planes cost NA (not p+1) registers each and the CTA runs
// XS times as many warps.  Rows are padded to whole warps (RPW = 32 / C rows per warp), so a warp never mixes parts.
template <int P, int CC, int XSPLIT>
struct MarchCfg {
    static constexpr int n = P + 1;
    static constexpr int C = CC;                          // real batch columns per CTA (NV = C / 4 complex vectors)
    static constexpr int NV = C / 4;
    static constexpr int XS = XSPLIT;
    static constexpr int NA = (n + XS - 1) / XS;
    static constexpr int RPW = 32 / C;
    static constexpr int WPH = (n + RPW - 1) / RPW;
    static constexpr int CWARPS = XS * WPH;
    static constexpr int THREADS = (CWARPS + 1) * 32;
    // stage layout: MAIN [n lines][P nodes][C] | FACE [n lines][C] (the x = P column) | R [P][P][C] | fields [P][P][4]
    static constexpr int FACE_OFF = n * P * C * 8;
    static constexpr int IN_BYTES = n * n * C * 8;
    __host__ __device__ static constexpr int ofs(int b, int a) { return a < P ? (b * P + a) * C : (n * P + b) * C; }   // doubles
    static constexpr int R_BYTES = P * P * C * 8;
    static constexpr int F_BYTES = P * P * 32;
    static constexpr int R_OFF = IN_BYTES;
    static constexpr int F_OFF = IN_BYTES + R_BYTES;
    static constexpr int STAGE_BYTES = ((F_OFF + F_BYTES + 127) / 128) * 128;
    static constexpr int STAGES = (200 * 1024 / STAGE_BYTES) < 8 ? (200 * 1024 / STAGE_BYTES) : 8;
    // FP32 product: a ring of NFB FP32 copies of the gathered plane (written by the converter warp) and the
    // per-thread FP64 pointwise store PW [P planes][P rows][P nodes][C] (recurrence terms stay FP64)
    static constexpr int NFB = 3;
    static constexpr int FB_BYTES = n * n * C * 4;
    static constexpr int PW_BYTES = P * P * P * C * 8;
    static constexpr int STAGES32_ = (200 * 1024 - PW_BYTES - NFB * FB_BYTES) / STAGE_BYTES;
    static constexpr int STAGES32 = STAGES32_ < 8 ? STAGES32_ : 8;
    // converter warps: fill the CTA up to whole groups of four warps (one per scheduler)
    static constexpr int NCW = 4 - (CWARPS + 1) % 4;
    static constexpr int THREADS32 = (CWARPS + 1 + NCW) * 32;
};

// Per-thread state of a consumer (part H of row j, lane = batch column).
template <int P, int CC, int XSPLIT, bool HASPH, int H, bool FULLV>
struct MarchConsumer {
    using Cfg = MarchCfg<P, CC, XSPLIT>;
    static constexpr int n = Cfg::n, C = Cfg::C, STAGES = Cfg::STAGES;
    static constexpr int A0 = H * Cfg::NA;
    static constexpr int NAH = (n - A0) < Cfg::NA ? (n - A0) : Cfg::NA;
    double acc[n][NAH];          // z-accumulators of the current cell: acc[k][ii], plane k, x-position A0 + ii
    double cin, cR, sg;          // W_y[j], P_y[j], F_y[j] are re-fetched from the constant bank where used
    double pAr, pAi, pBr, pBi;   // Bloch phase of this row's plain and x-face entries (HASPH)
    double* outcol;
    int j, col, s_spin, ri, ex, gy, g0;
    bool vok, jown, wy, xwrap, ywrap, valid, xph, yph;

    __device__ __forceinline__ void init(const StepConst& sc, const MarchArgs& ar, int row, int col_, int ex_, int ey,
                                         int chunk, int g0_, bool xw, bool yw) {
        valid = row < n;
        j = valid ? row : n - 1; col = col_; ex = ex_; g0 = g0_; xwrap = xw; ywrap = yw;
        xph = xw && ar.phd[0]; yph = yw && ar.phd[1];   // wraps that actually carry a phase
        s_spin = col / (C / 2); ri = col & 1;
        sg = ((ri == 0) != (s_spin == 0)) ? -1.0 : 1.0;
        const int vl = (col % (C / 2)) >> 1;
        const int v = chunk * Cfg::NV + vl;
        vok = valid && v < ar.nvec;
        jown = j < P;
        cin = (vok && ar.cin) ? __ldg(ar.cin + v) : 0.0;
        cR = (vok && ar.cR && ar.useR) ? __ldg(ar.cR + v) : 0.0;
        gy = ey * P + j; wy = gy == ar.n1[1]; if (wy) gy = 0;
        pAr = 1.0; pAi = 0.0;
        if (HASPH && wy) { pAr = ar.ph_re[1]; pAi = ar.ph_im[1]; }
        pBr = pAr; pBi = pAi;
        if (HASPH && xwrap) { pBr = pAr * ar.ph_re[0] - pAi * ar.ph_im[0]; pBi = pAr * ar.ph_im[0] + pAi * ar.ph_re[0]; }
        outcol = ar.out + ((long long)s_spin * ar.ld_out + (vok ? v : 0)) * 2 + ri;
#pragma unroll
        for (int k = 0; k < n; ++k)
#pragma unroll
            for (int ii = 0; ii < NAH; ++ii) acc[k][ii] = 0.0;
    }

    __device__ __forceinline__ static void phase_of(const MarchArgs& ar, bool wx, bool wyy, bool wz, double& pr, double& pi) {
        pr = 1.0; pi = 0.0;
        if (wx) { pr = ar.ph_re[0]; pi = ar.ph_im[0]; }
        if (wyy) { const double tt = pr * ar.ph_re[1] - pi * ar.ph_im[1]; pi = pr * ar.ph_im[1] + pi * ar.ph_re[1]; pr = tt; }
        if (wz) { const double tt = pr * ar.ph_re[2] - pi * ar.ph_im[2]; pi = pr * ar.ph_im[2] + pi * ar.ph_re[2]; pr = tt; }
    }

    // emit planes [0, nk) of the accumulators to global planes gzbase + k  (S3: one RED.ADD.F64 per node and column).
    // The REDs are left individually predicated on purpose: ptxas then spreads them between the FMAs of the
    // surrounding z-push; hoisting the predicate into one branch bunches 6(p+1) REDs together and costs 15 %.
    __device__ __forceinline__ void emit(const MarchArgs& ar, int gzbase, int nk) {
        const long long xsb = 32 * ar.ld_out;                          // bytes between consecutive nodes
        const long long x0 = (long long)ex * P + A0;
#pragma unroll
        for (int k = 0; k < n; ++k) {
            if (k < nk) {
                int gz = gzbase + k; const bool wz = gz == ar.n1[2]; if (wz) gz = 0;
                const bool anyw = xph | yph | (wz && ar.phd[2]);                  // CTA-uniform: interior CTAs skip the phase arithmetic
                double ar_ = pAr, ai_ = pAi, br_ = pBr, bi_ = pBi;      // conj-phase of plain / x-face columns of this row
                if (HASPH) {
                    if (wz) {
                        const double zr_ = ar.ph_re[2], zi_ = ar.ph_im[2];
                        const double t0 = ar_ * zr_ - ai_ * zi_; ai_ = ar_ * zi_ + ai_ * zr_; ar_ = t0;
                        const double t1 = br_ * zr_ - bi_ * zi_; bi_ = br_ * zi_ + bi_ * zr_; br_ = t1;
                    }
                    if (ri) { ai_ = -ai_; bi_ = -bi_; }
                }
                (void)ar_; (void)ai_; (void)br_; (void)bi_; (void)anyw;
                // running byte pointer along the x-line: two integer adds per RED instead of a full index computation
                char* line = reinterpret_cast<char*>(outcol) + ((long long)gz * ar.n1[1] + gy) * ar.n1[0] * xsb;
                char* pnode = line + x0 * xsb;
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) {
                    const bool wx = (A0 + ii == P) && xwrap;
                    double* dst = reinterpret_cast<double*>(wx ? line : pnode);
                    pnode += xsb;
                    double val = acc[k][ii];
                    if (HASPH && anyw) {
                        // times conj(phase), branch-free: (pr, pi) is (1, 0) where nothing wrapped
                        const double other = __shfl_xor_sync(0xffffffffu, val, 1);
                        const bool fc = A0 + ii == P;
                        val = fma(other, fc ? bi_ : ai_, val * (fc ? br_ : ar_));
                    }
                    if (FULLV) {
                        // every vector of the chunk exists (nvec % NV == 0): no predicate, so no branch around the RED
                        // (padding rows of a C = 16 warp add an exact zero)
                        atomicAdd(dst, (Cfg::RPW == 1 || valid) ? val : 0.0);
                    } else if (vok) {
                        atomicAdd(dst, val);
                    }
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
            // Bloch phase on wrapped entries (x: column a = P; y: row j = P; z: the wrapped plane), fixed up in place;
            // each part fixes its own x-positions of its row
            const bool wz = ar.phd[2] && (g0 + t) == ar.n1[2];
            if (xph | yph | wz) {                                        // CTA-uniform
                const bool wyy = yph && j == P;
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) {
                    const bool wx = xph && (A0 + ii == P);
                    const double val = IN[Cfg::ofs(j, A0 + ii) + col];
                    const double other = __shfl_xor_sync(0xffffffffu, val, 1);
                    if ((wx | wyy | wz) && valid) {
                        double pr, pi; phase_of(ar, wx, wyy, wz, pr, pi);
                        IN[Cfg::ofs(j, A0 + ii) + col] = ri == 0 ? val * pr - other * pi : other * pi + val * pr;
                    }
                }
                asm volatile("bar.sync 1, %0;" ::"r"(Cfg::CWARPS * 32) : "memory");   // consumer warps only
            }
        }
        const double* INc = IN + col;
        double row[n];
#pragma unroll
        for (int a = 0; a < n; ++a) row[a] = INc[Cfg::ofs(j, a)];
        double ip[NAH];
        // y-contraction: column A0 + ii of the plane against row j of KY
#pragma unroll
        for (int ii = 0; ii < NAH; ++ii) {
            double sy = 0.0;
#pragma unroll
            for (int b = 0; b < n; ++b) sy = fma(sc.KY[j][b], INc[Cfg::ofs(b, A0 + ii)], sy);
            ip[ii] = sc.WX[A0 + ii] * sy;
        }
        // x-contraction on the own row, own outputs
#pragma unroll
        for (int ii = 0; ii < NAH; ++ii) {
            double sx = 0.0;
#pragma unroll
            for (int a = 0; a < n; ++a) sx = fma(sc.KX[A0 + ii][a], row[a], sx);
            ip[ii] = fma(sc.WY[j], sx, ip[ii]);
        }
        double zr[NAH];
#pragma unroll
        for (int ii = 0; ii < NAH; ++ii) zr[ii] = sc.WX[A0 + ii] * (sc.WY[j] * row[A0 + ii]);
        if (lower) {
#pragma unroll
            for (int k = 0; k < n; ++k)
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) acc[k][ii] = fma(sc.KZ[k][P], zr[ii], acc[k][ii]);
#pragma unroll
            for (int ii = 0; ii < NAH; ++ii) acc[P][ii] = fma(sc.WZ[P], ip[ii], acc[P][ii]);
            // the previous cell is complete: emit its planes 0..P-1, carry its top plane over
            emit(ar, g0 + t - P, P);
#pragma unroll
            for (int ii = 0; ii < NAH; ++ii) acc[0][ii] = acc[P][ii];
#pragma unroll
            for (int k = 1; k < n; ++k)
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) acc[k][ii] = 0.0;
        }
        if (upper) {
            // z-push with the runtime cell-local index c: column c of KZ fetched from the constant bank
#pragma unroll
            for (int k = 0; k < n; ++k) {
                const double kz = sc.KZ[k][c];
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) acc[k][ii] = fma(kz, zr[ii], acc[k][ii]);
            }
            const double wzc = sc.WZ[c];
#pragma unroll
            for (int ii = 0; ii < NAH; ++ii) ip[ii] *= wzc;
            if (jown) {
                // S5 on the owned nodes of this plane (a < P): eq. 12 spin blocks, in-term, R-term
                const double pz = sc.PZ[c] * sc.PY[j], fz = sc.FZ[c] * sc.FY[j] * cin;
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) {
                    const int a = A0 + ii;
                    if (a < P) {
                        // (B_x -+ i B_y) u_other: real part B_x u_re +- B_y u_im, imaginary part B_x u_im -+ B_y u_re, i.e.
                        // B_x * (other spin, same part) + sg * B_y * (other spin, other part), sg fixed per thread
                        const double in_own = row[a];
                        const double o_same = INc[Cfg::ofs(j, a) + ((col ^ (C / 2)) - col)];
                        const double o_flip = INc[Cfg::ofs(j, a) + ((col ^ (C / 2 + 1)) - col)];
                        const double diag = Fs[(j * P + a) * 4 + s_spin];
                        const double2 bxy = *reinterpret_cast<const double2*>(Fs + (j * P + a) * 4 + 2);
                        const double pot = fma(diag, in_own, fma(bxy.x, o_same, (sg * bxy.y) * o_flip));
                        double val = fma(pz * sc.PX[a], pot, ip[ii]);
                        val = fma(fz * sc.FX[a], in_own, val);
                        if (ar.useR) val = fma(cR, Rs[(j * P + a) * C + col], val);
                        ip[ii] = val;
                    }
                }
            }
            // add the in-plane + pointwise part to the accumulator of the plane's own index
#pragma unroll
            for (int k = 0; k < P; ++k) {
                if (c == k) {
#pragma unroll
                    for (int ii = 0; ii < NAH; ++ii) acc[k][ii] += ip[ii];
                }
            }
        }
        __syncwarp();
        if ((threadIdx.x & 31) == 0) mbar_arrive(&empty_bar[s]);
    }

    __device__ __forceinline__ void run(const StepConst& sc, const MarchArgs& ar, unsigned char* smem, uint64_t* full_bar,
                                        uint64_t* empty_bar, int T) {
        int c = 0;
#pragma unroll 1
        for (int t = 0; t < T; ++t) {
            plane(sc, ar, smem, full_bar, empty_bar, t, c, c == 0 && t > 0, t < T - 1);
            c = (c + 1 == P) ? 0 : c + 1;
        }
        emit(ar, g0 + T - 1, 1);                                   // partial of the segment's top face
    }
};

// ---------------------------------------------------------------------------------------------
// FP32 product (CHFSI_FP32): the Laplacian of fl32(in) is computed and accumulated in FP32 from
// the converter warp's FP32 copy of the plane; the pointwise potential, the in-term and the R-term of eq. 11 are
// computed in FP64 from the FP64 stage and parked in the thread's own slots of PW until the cell is emitted, where
// the FP32 Laplacian is widened exactly, scaled by cH in FP64 and both are sent out with one RED.ADD.F64.
template <int P, int CC, int XSPLIT, bool HASPH, int H, bool FULLV>
struct MarchConsumerF32 {
    using Cfg = MarchCfg<P, CC, XSPLIT>;
    static constexpr int n = Cfg::n, C = Cfg::C, STAGES = Cfg::STAGES32, NFB = Cfg::NFB;
    static constexpr int A0 = H * Cfg::NA;
    static constexpr int NAH = (n - A0) < Cfg::NA ? (n - A0) : Cfg::NA;
    float acc[n][NAH];
    float kyrow[n], wxy[NAH];
    float wyj;
    double pyj, fyj, cin, cR, sg;
    double pAr, pAi, pBr, pBi;
    double* outcol;
    double* pw;                  // PW + (j * P) * C + col : this thread's pointwise slots, [c][.][a][.]
    int j, col, s_spin, ri, ex, gy, g0;
    bool vok, jown, wy, xwrap, ywrap, valid, xph, yph;

    __device__ __forceinline__ void init(const StepConst& sc, const MarchArgs& ar, double* PW, int row, int col_, int ex_, int ey,
                                         int chunk, int g0_, bool xw, bool yw) {
        valid = row < n;
        j = valid ? row : n - 1; col = col_; ex = ex_; g0 = g0_; xwrap = xw; ywrap = yw;
        xph = xw && ar.phd[0]; yph = yw && ar.phd[1];   // wraps that actually carry a phase
        s_spin = col / (C / 2); ri = col & 1;
        sg = ((ri == 0) != (s_spin == 0)) ? -1.0 : 1.0;
        const int vl = (col % (C / 2)) >> 1;
        const int v = chunk * Cfg::NV + vl;
        vok = valid && v < ar.nvec;
        jown = j < P;
#pragma unroll
        for (int b = 0; b < n; ++b) kyrow[b] = sc.KYf[j][b];
#pragma unroll
        for (int ii = 0; ii < NAH; ++ii) wxy[ii] = sc.WXf[A0 + ii] * sc.WYf[j];
        wyj = sc.WYf[j]; pyj = sc.PY[j]; fyj = sc.FY[j];
        cin = (vok && ar.cin) ? __ldg(ar.cin + v) : 0.0;
        cR = (vok && ar.cR && ar.useR) ? __ldg(ar.cR + v) : 0.0;
        gy = ey * P + j; wy = gy == ar.n1[1]; if (wy) gy = 0;
        pAr = 1.0; pAi = 0.0;
        if (HASPH && wy) { pAr = ar.ph_re[1]; pAi = ar.ph_im[1]; }
        pBr = pAr; pBi = pAi;
        if (HASPH && xwrap) { pBr = pAr * ar.ph_re[0] - pAi * ar.ph_im[0]; pBi = pAr * ar.ph_im[0] + pAi * ar.ph_re[0]; }
        outcol = ar.out + ((long long)s_spin * ar.ld_out + (vok ? v : 0)) * 2 + ri;
        pw = PW + (jown ? j : 0) * P * C + col;
#pragma unroll
        for (int k = 0; k < n; ++k)
#pragma unroll
            for (int ii = 0; ii < NAH; ++ii) acc[k][ii] = 0.f;
    }

    __device__ __forceinline__ static void phase_of(const MarchArgs& ar, bool wx, bool wyy, bool wz, double& pr, double& pi) {
        pr = 1.0; pi = 0.0;
        if (wx) { pr = ar.ph_re[0]; pi = ar.ph_im[0]; }
        if (wyy) { const double tt = pr * ar.ph_re[1] - pi * ar.ph_im[1]; pi = pr * ar.ph_im[1] + pi * ar.ph_re[1]; pr = tt; }
        if (wz) { const double tt = pr * ar.ph_re[2] - pi * ar.ph_im[2]; pi = pr * ar.ph_im[2] + pi * ar.ph_re[2]; pr = tt; }
    }

    // emit planes [0, nk): out += cH * (double)acc + PW (owned nodes only; with_pw false for the segment's top face)
    __device__ __forceinline__ void emit(const StepConst& sc, const MarchArgs& ar, int gzbase, int nk, bool with_pw) {
        const long long xsb = 32 * ar.ld_out;                          // bytes between consecutive nodes
        const long long x0 = (long long)ex * P + A0;
#pragma unroll
        for (int k = 0; k < n; ++k) {
            if (k < nk) {
                int gz = gzbase + k; const bool wz = gz == ar.n1[2]; if (wz) gz = 0;
                const bool anyw = xph | yph | (wz && ar.phd[2]);                  // CTA-uniform: interior CTAs skip the phase arithmetic
                double ar_ = pAr, ai_ = pAi, br_ = pBr, bi_ = pBi;      // conj-phase of plain / x-face columns of this row
                if (HASPH) {
                    if (wz) {
                        const double zr_ = ar.ph_re[2], zi_ = ar.ph_im[2];
                        const double t0 = ar_ * zr_ - ai_ * zi_; ai_ = ar_ * zi_ + ai_ * zr_; ar_ = t0;
                        const double t1 = br_ * zr_ - bi_ * zi_; bi_ = br_ * zi_ + bi_ * zr_; br_ = t1;
                    }
                    if (ri) { ai_ = -ai_; bi_ = -bi_; }
                }
                (void)ar_; (void)ai_; (void)br_; (void)bi_; (void)anyw;
                // running byte pointer along the x-line: two integer adds per RED instead of a full index computation
                char* line = reinterpret_cast<char*>(outcol) + ((long long)gz * ar.n1[1] + gy) * ar.n1[0] * xsb;
                char* pnode = line + x0 * xsb;
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) {
                    const bool wx = (A0 + ii == P) && xwrap;
                    double* dst = reinterpret_cast<double*>(wx ? line : pnode);
                    pnode += xsb;
                    double val = sc.cH * (double)acc[k][ii];
                    if (A0 + ii < P && k < P) {
                        if (with_pw && jown) val += pw[(k * P * P + A0 + ii) * C];
                    }
                    if (HASPH && anyw) {
                        // times conj(phase), branch-free: (pr, pi) is (1, 0) where nothing wrapped
                        const double other = __shfl_xor_sync(0xffffffffu, val, 1);
                        const bool fc = A0 + ii == P;
                        val = fma(other, fc ? bi_ : ai_, val * (fc ? br_ : ar_));
                    }
                    if (FULLV) {
                        // every vector of the chunk exists (nvec % NV == 0): no predicate, so no branch around the RED
                        // (padding rows of a C = 16 warp add an exact zero)
                        atomicAdd(dst, (Cfg::RPW == 1 || valid) ? val : 0.0);
                    } else if (vok) {
                        atomicAdd(dst, val);
                    }
                }
            }
        }
    }

    __device__ __forceinline__ void plane(const StepConst& sc, const MarchArgs& ar, unsigned char* smem, const float* FBbase,
                                          uint64_t* full_bar, uint64_t* empty_bar, uint64_t* cfull_bar, uint64_t* cempty_bar,
                                          int t, int c, bool lower, bool upper) {
        const int s = t % STAGES, f = t % NFB;
        mbar_wait(&cfull_bar[f], (t / NFB) & 1);
        mbar_wait(&full_bar[s], (t / STAGES) & 1);           // already complete; orders this thread after the TMA writes
        const double* INc = reinterpret_cast<const double*>(smem + (size_t)s * Cfg::STAGE_BYTES) + col;
        const double* Rs = reinterpret_cast<const double*>(smem + (size_t)s * Cfg::STAGE_BYTES + Cfg::R_OFF);
        const double* Fs = reinterpret_cast<const double*>(smem + (size_t)s * Cfg::STAGE_BYTES + Cfg::F_OFF);
        const float* FBc = FBbase + (size_t)f * (Cfg::FB_BYTES / 4) + col;
        float row[n];
#pragma unroll
        for (int a = 0; a < n; ++a) row[a] = FBc[Cfg::ofs(j, a)];
        float ip[NAH];
#pragma unroll
        for (int ii = 0; ii < NAH; ++ii) {
            float sy = 0.f;
#pragma unroll
            for (int b = 0; b < n; ++b) sy = fmaf(kyrow[b], FBc[Cfg::ofs(b, A0 + ii)], sy);
            ip[ii] = sc.WXf[A0 + ii] * sy;
        }
#pragma unroll
        for (int ii = 0; ii < NAH; ++ii) {
            float sx = 0.f;
#pragma unroll
            for (int a = 0; a < n; ++a) sx = fmaf(sc.KXf[A0 + ii][a], row[a], sx);
            ip[ii] = fmaf(wyj, sx, ip[ii]);
        }
        float zr[NAH];
#pragma unroll
        for (int ii = 0; ii < NAH; ++ii) zr[ii] = wxy[ii] * row[A0 + ii];
        if (lower) {
#pragma unroll
            for (int k = 0; k < n; ++k)
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) acc[k][ii] = fmaf(sc.KZf[k][P], zr[ii], acc[k][ii]);
#pragma unroll
            for (int ii = 0; ii < NAH; ++ii) acc[P][ii] = fmaf(sc.WZf[P], ip[ii], acc[P][ii]);
            emit(sc, ar, g0 + t - P, P, true);
#pragma unroll
            for (int ii = 0; ii < NAH; ++ii) acc[0][ii] = acc[P][ii];
#pragma unroll
            for (int k = 1; k < n; ++k)
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) acc[k][ii] = 0.f;
        }
        if (upper) {
#pragma unroll
            for (int k = 0; k < n; ++k) {
                const float kz = sc.KZf[k][c];
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) acc[k][ii] = fmaf(kz, zr[ii], acc[k][ii]);
            }
            const float wzc = sc.WZf[c];
#pragma unroll
            for (int k = 0; k < P; ++k) {
                if (c == k) {
#pragma unroll
                    for (int ii = 0; ii < NAH; ++ii) acc[k][ii] = fmaf(wzc, ip[ii], acc[k][ii]);
                }
            }
            if (jown) {
                // S5 in FP64 on the owned nodes of this plane: eq. 12 spin blocks, in-term, R-term -> PW[c][j][a]
                const double pz = sc.PZ[c] * pyj, fz = sc.FZ[c] * fyj * cin;
                double* pwc = pw + c * P * P * C;
#pragma unroll
                for (int ii = 0; ii < NAH; ++ii) {
                    const int a = A0 + ii;
                    if (a < P) {
                        const double in_own = INc[Cfg::ofs(j, a)];
                        const double o_same = INc[Cfg::ofs(j, a) + ((col ^ (C / 2)) - col)];
                        const double o_flip = INc[Cfg::ofs(j, a) + ((col ^ (C / 2 + 1)) - col)];
                        const double diag = Fs[(j * P + a) * 4 + s_spin];
                        const double2 bxy = *reinterpret_cast<const double2*>(Fs + (j * P + a) * 4 + 2);
                        double val = (pz * sc.PX[a]) * fma(diag, in_own, fma(bxy.x, o_same, (sg * bxy.y) * o_flip));
                        val = fma(fz * sc.FX[a], in_own, val);
                        if (ar.useR) val = fma(cR, Rs[(j * P + a) * C + col], val);
                        pwc[a * C] = val;
                    }
                }
            }
        }
        __syncwarp();
        if ((threadIdx.x & 31) == 0) { mbar_arrive(&empty_bar[s]); mbar_arrive(&cempty_bar[f]); }
    }

    __device__ __forceinline__ void run(const StepConst& sc, const MarchArgs& ar, unsigned char* smem, const float* FBbase,
                                        uint64_t* full_bar, uint64_t* empty_bar, uint64_t* cfull_bar, uint64_t* cempty_bar, int T) {
        int c = 0;
#pragma unroll 1
        for (int t = 0; t < T; ++t) {
            plane(sc, ar, smem, FBbase, full_bar, empty_bar, cfull_bar, cempty_bar, t, c, c == 0 && t > 0, t < T - 1);
            c = (c + 1 == P) ? 0 : c + 1;
        }
        emit(sc, ar, g0 + T - 1, 1, false);
    }
};

// Converter warp of the FP32 product: fl32 of the gathered plane (one RN cast per value, north_star (5): conversion
// fused into the load path), with the Bloch phase of wrapped entries applied in FP64 before the cast.
template <int P, int CC, int XSPLIT, bool HASPH>
__device__ __forceinline__ void march_convert(const MarchArgs& ar, unsigned char* smem, float* FBbase, uint64_t* full_bar,
                                              uint64_t* cfull_bar, uint64_t* cempty_bar, int cw, int lane, int g0, int T,
                                              bool xwrap, bool ywrap, double isc) {
    using Cfg = MarchCfg<P, CC, XSPLIT>;
    constexpr int n = Cfg::n, C = Cfg::C, STAGES = Cfg::STAGES32, NFB = Cfg::NFB, HC = C / 2;
#pragma unroll 1
    for (int t = 0; t < T; ++t) {
        const int s = t % STAGES, f = t % NFB;
        mbar_wait(&cempty_bar[f], ((t / NFB) & 1) ^ 1);
        mbar_wait(&full_bar[s], (t / STAGES) & 1);
        const double2* IN2 = reinterpret_cast<const double2*>(smem + (size_t)s * Cfg::STAGE_BYTES);
        float2* FB2 = reinterpret_cast<float2*>(FBbase + (size_t)f * (Cfg::FB_BYTES / 4));
        const bool wz = HASPH && ar.phd[2] && (g0 + t) == ar.n1[2];
#pragma unroll 4
        for (int e = cw * 32 + lane; e < n * n * HC; e += 32 * Cfg::NCW) {
            double2 v = IN2[e];
            if (HASPH) {
                const int sl = e / HC;                               // slot: MAIN [b][a < P] then FACE [b]
                const bool face = sl >= n * P;
                const int b = face ? sl - n * P : sl / P;
                const bool wx = xwrap && face, wyy = ywrap && b == P;
                if (wx | wyy | wz) {
                    double pr = 1.0, pi = 0.0;
                    if (wx) { pr = ar.ph_re[0]; pi = ar.ph_im[0]; }
                    if (wyy) { const double tt = pr * ar.ph_re[1] - pi * ar.ph_im[1]; pi = pr * ar.ph_im[1] + pi * ar.ph_re[1]; pr = tt; }
                    if (wz) { const double tt = pr * ar.ph_re[2] - pi * ar.ph_im[2]; pi = pr * ar.ph_im[2] + pi * ar.ph_re[2]; pr = tt; }
                    v = make_double2(v.x * pr - v.y * pi, v.x * pi + v.y * pr);
                }
            }
            FB2[e] = make_float2((float)(v.x * isc), (float)(v.y * isc));   // isc: exact power-of-two rescaling
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&cfull_bar[f]);
    }
}

template <int P, int CC, int XSPLIT, bool HASPH, int H, bool FULLV>
__device__ __forceinline__ void march_consume(const StepConst& sc, const MarchArgs& ar, unsigned char* smem, uint64_t* full_bar,
                                           uint64_t* empty_bar, int row, int col, int ex, int ey, int chunk, int g0, int T,
                                           bool xwrap, bool ywrap) {
    MarchConsumer<P, CC, XSPLIT, HASPH, H, FULLV> cs;
    cs.init(sc, ar, row, col, ex, ey, chunk, g0, xwrap, ywrap);
    cs.run(sc, ar, smem, full_bar, empty_bar, T);
}

template <int P, int CC, int XSPLIT, bool HASPH, int H, bool FULLV>
__device__ __forceinline__ void march_consume32(const StepConst& sc, const MarchArgs& ar, unsigned char* smem, float* FB, double* PW,
                                                uint64_t* full_bar, uint64_t* empty_bar, uint64_t* cfull_bar, uint64_t* cempty_bar,
                                                int row, int col, int ex, int ey, int chunk, int g0, int T, bool xwrap, bool ywrap) {
    MarchConsumerF32<P, CC, XSPLIT, HASPH, H, FULLV> cs;
    cs.init(sc, ar, PW, row, col, ex, ey, chunk, g0, xwrap, ywrap);
    cs.run(sc, ar, smem, FB, full_bar, empty_bar, cfull_bar, cempty_bar, T);
}

template <int P, int CC, int XSPLIT, bool HASPH, bool F32, bool FULLV>
__global__ void __launch_bounds__(F32 ? MarchCfg<P, CC, XSPLIT>::THREADS32 : MarchCfg<P, CC, XSPLIT>::THREADS, 1)
cell_march_kernel(const __grid_constant__ StepConst sc, const __grid_constant__ MarchArgs ar,
                  const __grid_constant__ MarchMaps mp) {
    using Cfg = MarchCfg<P, CC, XSPLIT>;
    constexpr int n = Cfg::n, C = Cfg::C, STAGES = F32 ? Cfg::STAGES32 : Cfg::STAGES, NFB = Cfg::NFB;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full_bar[STAGES], empty_bar[STAGES], cfull_bar[NFB], cempty_bar[NFB];
    float* FB = reinterpret_cast<float*>(smem + (size_t)STAGES * Cfg::STAGE_BYTES);
    double* PW = reinterpret_cast<double*>(smem + (size_t)STAGES * Cfg::STAGE_BYTES + NFB * Cfg::FB_BYTES);
    (void)n; (void)FB; (void)PW;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // blockIdx -> (ex fastest, ey, seg, chunk): neighbours in x/y run together, so shared faces hit in L2
    // With C = 16 a 128-byte line holds the rows of TWO chunks: the pair runs side by side (pair index fastest).
    int bid = blockIdx.x;
    int cpair = 0;
    if (C == 16) { cpair = bid & 1; bid >>= 1; }
    const int ex = bid % ar.nc[0]; bid /= ar.nc[0];
    const int ey = bid % ar.nc[1]; bid /= ar.nc[1];
    const int seg = bid % ar.nseg;
    const int chunk = C == 16 ? 2 * (bid / ar.nseg) + cpair : bid / ar.nseg;
    if (chunk >= ar.nchunks) return;              // odd chunk count: the last pair is half empty
    const int T = ar.cps * P + 1;                 // planes this CTA marches through
    const int g0 = seg * ar.cps * P;              // first global plane
    const bool xwrap = ex == ar.nc[0] - 1, ywrap = ey == ar.nc[1] - 1;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], Cfg::CWARPS); }
        for (int f = 0; f < NFB; ++f) { mbar_init(&cfull_bar[f], Cfg::NCW); mbar_init(&cempty_bar[f], Cfg::CWARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == Cfg::CWARPS) {
        // ================================ producer ================================
        if (lane == 0) {
            const int col0 = chunk * (C / 2);                     // doubles
            uint64_t pol_last;
            asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_last));
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
                // lines ey*P .. ey*P+P of plane gz; the last one wraps to y = 0 in the last cell row
                const int line = gz * ar.n1[1] + ey * P;
                const int xr = 2 * ex * P;                                  // first (node, spin) row of the cell in its x-line
                const int xf = xwrap ? 0 : xr + 2 * P;                       // rows of the x = P face column
                if (!ywrap) {
                    tma_load_3d(st, &mp.main[0], col0, xr, line, &full_bar[s]);
                    tma_load_3d(st + Cfg::FACE_OFF, &mp.face[0], col0, xf, line, &full_bar[s]);
                } else {
                    tma_load_3d(st, &mp.main[1], col0, xr, line, &full_bar[s]);
                    tma_load_3d(st + P * P * C * 8, &mp.main[2], col0, xr, gz * ar.n1[1], &full_bar[s]);
                    tma_load_3d(st + Cfg::FACE_OFF, &mp.face[1], col0, xf, line, &full_bar[s]);
                    tma_load_3d(st + Cfg::FACE_OFF + P * C * 8, &mp.face[2], col0, xf, gz * ar.n1[1], &full_bar[s]);
                }
                if (owned) {
                    if (ar.useR) tma_load_3d(st + Cfg::R_OFF, &mp.R, col0, xr, line, &full_bar[s]);
                    tma_load_2d_hint(st + Cfg::F_OFF, &mp.F, 4 * ex * P, line, &full_bar[s], pol_last);
                }
            }
        }
        return;
    }

    if (F32 && warp > Cfg::CWARPS) {
        march_convert<P, CC, XSPLIT, HASPH>(ar, smem, FB, full_bar, cfull_bar, cempty_bar, warp - Cfg::CWARPS - 1, lane, g0, T,
                                            xwrap && ar.phd[0], ywrap && ar.phd[1], sc.in_scale);
        return;
    }

    // ================================ consumers ================================
    const int h = warp / Cfg::WPH;
    const int row = (warp % Cfg::WPH) * Cfg::RPW + lane / C;
    const int col = lane % C;
    (void)h; (void)row;
#define MARCH_PART(HH)                                                                                              \
    if (HH < XSPLIT && h == HH) {                                                                                   \
        if (F32)                                                                                                    \
            march_consume32<P, CC, XSPLIT, HASPH, (HH < XSPLIT ? HH : 0), FULLV>(sc, ar, smem, FB, PW, full_bar, empty_bar, \
                                                                          cfull_bar, cempty_bar, row, col, ex, ey,  \
                                                                          chunk, g0, T, xwrap, ywrap);              \
        else                                                                                                        \
            march_consume<P, CC, XSPLIT, HASPH, (HH < XSPLIT ? HH : 0), FULLV>(sc, ar, smem, full_bar, empty_bar, row, col, ex, ey, \
                                                                        chunk, g0, T, xwrap, ywrap);               \
    }
    MARCH_PART(0) MARCH_PART(1) MARCH_PART(2)
#undef MARCH_PART
}

bool march_supported(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a) {
    if (prec != CHFSI_FP64 && prec != CHFSI_FP32) return false;
    if (m->p != 2 && m->p != 4 && m->p != 6 && m->p != 8) return false;
    if (m->dF == nullptr) return false;
    // TMA needs 16-byte aligned bases/strides (always true for complex128 rows) and 32-bit row coordinates
    if (2 * m->nnodes >= (1ll << 31)) return false;
    if (m->mc.n1[0] * 4ll * 8 % 16 != 0) return false;
    if (((uintptr_t)a.in & 15) || ((uintptr_t)a.out & 15) || (a.R && ((uintptr_t)a.R & 15))) return false;
    return get_encode() != nullptr;
}

static void build_step_const(const chfsi_mesh* m, const CellArgs& a, StepConst& sc) {
    const MeshConst& mc = m->mc;
    const int n = mc.n;
    const bool sin_ = (a.flags & kScaleIn) != 0, sout_ = (a.flags & kSoutInvM) != 0, massin = (a.flags & kMassIn) != 0;
    std::memset(&sc, 0, sizeof(sc));
    const double isc = a.in_scale > 0.0 ? a.in_scale : 1.0;        // used by the FP32 product only
    sc.cH = a.cH / isc;
    sc.in_scale = isc;
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
                (d == 0 ? sc.KXf : d == 1 ? sc.KYf : sc.KZf)[i][b] = (float)(so * mc.Kd[d][i][b] * sb);
            }
            W[i] = mc.w[i] * so * si;
            (d == 0 ? sc.WXf : d == 1 ? sc.WYf : sc.WZf)[i] = (float)W[i];
            const double fu = sin_ ? 1.0 : mc.m1[d][i];                // u = m w: Z-form u = in, else m * in
            Pp[i] = so * fu * (d == 0 ? a.cH : 1.0);
            Fp[i] = massin ? mc.m1[d][i] : 1.0;
        }
    }
}

template <int P, int CC, int XSPLIT, bool F32>
static cudaError_t launch_march_t(const chfsi_mesh* m, const CellArgs& a, cudaStream_t st) {
    using Cfg = MarchCfg<P, CC, XSPLIT>;
    StepConst sc;
    build_step_const(m, a, sc);
    MarchArgs ar;
    std::memset(&ar, 0, sizeof(ar));
    for (int d = 0; d < 3; ++d) {
        ar.nc[d] = m->mc.nc[d]; ar.n1[d] = m->mc.n1[d];
        ar.ph_re[d] = m->mc.ph_re[d]; ar.ph_im[d] = m->mc.ph_im[d];
    }
    ar.has_phase = m->mc.has_phase;
    for (int d = 0; d < 3; ++d) ar.phd[d] = (m->mc.ph_re[d] != 1.0 || m->mc.ph_im[d] != 0.0) ? 1 : 0;
    ar.nvec = a.nvec; ar.nchunks = (a.nvec + Cfg::NV - 1) / Cfg::NV;
    ar.useR = (a.R != nullptr && a.cR != nullptr) ? 1 : 0;
    ar.fields = m->dF; ar.cin = a.cin; ar.cR = a.cR; ar.out = a.out; ar.ld_out = a.ld_out;
    // z segmentation: enough CTAs for >= ~4 waves of one CTA per SM
    const long long base = (long long)ar.nc[0] * ar.nc[1] * ar.nchunks;
    int nseg = 1;
    for (int cand = 1; cand <= ar.nc[2]; ++cand)
        if (ar.nc[2] % cand == 0) { nseg = cand; if (base * cand >= 4 * 148) break; }
    ar.nseg = nseg; ar.cps = ar.nc[2] / nseg;
    MarchMaps mp;
    constexpr int BC = CC / 2;
    const int nl[3] = {P + 1, P, 1};
    for (int i = 0; i < 3; ++i)
        if (!make_map3(&mp.main[i], m, a.in, a.ld_in, a.nvec, BC, 2 * P, nl[i]) || !make_map3(&mp.face[i], m, a.in, a.ld_in, a.nvec, BC, 2, nl[i]))
            return cudaErrorInvalidValue;
    if (!make_map3(&mp.R, m, ar.useR ? a.R : a.in, ar.useR ? a.ld_R : a.ld_in, a.nvec, BC, 2 * P, P) || !make_mapF(&mp.F, m, P))
        return cudaErrorInvalidValue;
    const size_t smem = F32 ? (size_t)Cfg::STAGES32 * Cfg::STAGE_BYTES + Cfg::NFB * Cfg::FB_BYTES + Cfg::PW_BYTES
                            : (size_t)Cfg::STAGES * Cfg::STAGE_BYTES;
    static bool attr_done[128] = {false};   // per template instantiation
    const bool full = (a.nvec % Cfg::NV) == 0;          // every CTA's vector tile is complete: unpredicated REDs
    auto kern = m->mc.has_phase ? (full ? cell_march_kernel<P, CC, XSPLIT, true, F32, true> : cell_march_kernel<P, CC, XSPLIT, true, F32, false>)
                                : (full ? cell_march_kernel<P, CC, XSPLIT, false, F32, true> : cell_march_kernel<P, CC, XSPLIT, false, F32, false>);
    const int slot = (m->device & 31) * 4 + (m->mc.has_phase ? 2 : 0) + (full ? 1 : 0);
    if (!attr_done[slot]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_done[slot] = true;
    }
    const long long grid = CC == 16 ? (long long)ar.nc[0] * ar.nc[1] * nseg * 2 * ((ar.nchunks + 1) / 2) : base * nseg;
    kern<<<(unsigned)grid, F32 ? Cfg::THREADS32 : Cfg::THREADS, smem, st>>>(sc, ar, mp);
    return cudaGetLastError();
}

cudaError_t launch_cell_march(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t st) {
    const bool f32 = prec == CHFSI_FP32;
    switch (m->p) {
        case 2: return f32 ? launch_march_t<2, 32, 1, true>(m, a, st) : launch_march_t<2, 32, 1, false>(m, a, st);
        case 4: return f32 ? launch_march_t<4, 32, 1, true>(m, a, st) : launch_march_t<4, 32, 1, false>(m, a, st);
        case 6: return f32 ? launch_march_t<6, 32, 1, true>(m, a, st) : launch_march_t<6, 32, 1, false>(m, a, st);
        case 8: return f32 ? launch_march_t<8, 16, 1, true>(m, a, st) : launch_march_t<8, 16, 2, false>(m, a, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace chfsi
