// Line-owned x/y/z cell kernel: the dominant kernel of the filter on sm_100a (S1, S2, S3, S5, S6 of DESIGN.md in one pass).
//
// One CTA owns the xy-footprint of one FE cell column (ex, ey), a z-segment of `cps` cells and C real batch columns
// (NV = C/4 complex vectors: re/im of both spin components, which the real spin-diagonal Laplacian treats alike), and
// marches through the xy-planes of that column:
//   producer warp : one elected lane streams each plane -- the (p+1)^2 gathered node rows of `in`, the p^2 owned rows of
//                   R and the packed local fields -- into a ring of shared-memory stages with TMA
//                   (cp.async.bulk.tensor.3d, completing on mbarriers).  S1 gather, PAPER.md:204 (i).
//   consumer warps: a thread is (index q, batch column); q plays two roles in the two phases of a plane:
//     X-phase : q = footprint row j.  The thread holds the whole x-line (p+1 values, p+1 LDS) and produces all p+1
//               outputs of the x-contraction with the even/odd decomposition of the centrosymmetric 1-D matrix
//               ("even/odd decomposition ... halves the multiplication count"), and parks them in a
//               double-buffered shared-memory plane XR.  The Bloch phase of wrapped entries is fixed up here.
//     YZ-phase: q = x-position a.  The thread holds the whole y-line at its x-position (p+1 LDS), does the y-contraction
//               even/odd in registers, adds the x-part from XR, and *pushes* the line into the (p+1) x (p+1)
//               z-accumulators acc[k][j] of the current cell that it keeps in registers: the z-contraction never touches
//               memory and z-faces are assembled in registers (the top plane carries over to the next cell).
//               The 2x2 spin potential (eq. 12), the in-term and the R-term of eq. 11 (S5) are added to the accumulator of
//               the node's own plane.  When a cell completes, its p planes leave with one RED.ADD per node and column
//               (S3, PAPER.md:204 (iii)).
// Every load of the contractions is a full line owned by the thread that uses it: (p+1) shared-memory loads feed
// ~(p+1)^2/2 + (p+1) arithmetic instructions, instead of one load per FMA in a row-owned y-contraction.
// Precision modes (template MODE):
//   M_F64  : in / out / R complex128, FP64 arithmetic                                  (CHFSI_FP64)
//   M_F32P : in / out / R complex128; in is rounded to FP32 on load, the Laplacian is contracted and accumulated in FP32,
//            widened at emission; pointwise + recurrence terms stay FP64 and leave with their own RED (CHFSI_FP32)
//   M_F32S : in / out complex64 (FP32-stored multivectors), R complex128; FP32 arithmetic, the R-term is
//            formed in FP64 and rounded once                                            (CHFSI_FP32_STORED)
#include <cuda.h>

#include <cmath>
#include <cstring>
#include <mutex>

#include "chfsi_internal.h"
#include "tma_util.cuh"

namespace chfsi {

enum XyzMode : int { M_F64 = 0, M_F32P = 1, M_F32S = 2 };

template <int MODE> struct ModeT;
template <> struct ModeT<M_F64> { using TI = double; using TC = double; using TO = double; };
template <> struct ModeT<M_F32P> { using TI = double; using TC = float; using TO = double; };
template <> struct ModeT<M_F32S> { using TI = float; using TC = float; using TO = float; };

// even/odd tables of a centrosymmetric (p+1)x(p+1) matrix K (p even, H = p/2 pairs (q, p-q), middle index p/2):
//   E_q = sum_{b<H} A[q][b] (v_b + v_{p-b}) + Am[q] v_mid ,  O_q = sum_{b<H} B[q][b] (v_b - v_{p-b}) ,
//   (K v)_q = E_q + O_q ,  (K v)_{p-q} = E_q - O_q  (q < H) ;  (K v)_mid = sum_{b<H} Mid[b] (v_b + v_{p-b}) + Mid[H] v_mid
template <typename TC>
struct EoTab { TC A[4][4]; TC Am[4]; TC B[4][4]; TC Mid[5]; };

template <typename TC>
struct XyzConst {
    EoTab<TC> X, Y;             // all scalings folded in, see build_const
    TC KZ[kMaxN][kMaxN];
    TC WX[kMaxN], WY[kMaxN], WZ[kMaxN];
    double M1X[kMaxN], M1Y[kMaxN], M1Z[kMaxN];   // 1-D mass factors (MASSIN launches: the residual S0)
    double cHp;                 // coefficient of the potential term
    double cH;                  // FP32 product: step coefficient / in_scale, applied where the FP32 Laplacian leaves
    double in_scale;            // FP32 product: power of two applied (in FP64) to `in` before the cast
};

// Rows of the footprint owned by half JH of a thread pair: whole even/odd pairs (q, P - q), so that each half computes
// its outputs of the 1-D contractions with the even/odd decomposition.  Local index l -> row(l).
template <int P, int JH>
struct RowSet {
    static constexpr int H = P / 2, MID = P / 2;
    static constexpr int NP0 = (H + 1) / 2;
    static constexpr int NPAIR = JH == 0 ? NP0 : H - NP0;
    static constexpr int Q0 = JH == 0 ? 0 : NP0;
    static constexpr bool HASMID = (JH == 0) == (H % 2 == 0);
    static constexpr int NJ = 2 * NPAIR + (HASMID ? 1 : 0);
    __host__ __device__ static constexpr int row(int l) { return l == 2 * NPAIR ? MID : (l % 2 == 0 ? Q0 + l / 2 : P - (Q0 + l / 2)); }
};

template <int P, int CC, int MODE>
struct XyzCfg {
    using TI = typename ModeT<MODE>::TI;
    using TC = typename ModeT<MODE>::TC;
    static constexpr int n = P + 1, C = CC, NV = C / 4;
    static constexpr int RPW = 32 / C;                       // indices q per warp
    static constexpr int NQW = (n + RPW - 1) / RPW;          // warps per half
    static constexpr int NCW = 2 * NQW;                      // consumer warps (two halves of the rows)
    static constexpr int THREADS = (NCW + 1) * 32;
    // stage: MAIN [n lines][P nodes][C] | FACE [n lines][C] (the x = P column) | R [P][P][C] f64 | fields [P][P][4] f64
    static constexpr int FACE_OFF = n * P * C * (int)sizeof(TI);
    static constexpr int IN_BYTES = n * n * C * (int)sizeof(TI);
    static constexpr int R_BYTES = P * P * C * 8;
    static constexpr int F_BYTES = P * P * (MODE == M_F32S ? 16 : 32);   // FP32-stored: the FP32 copy of the fields
    static constexpr int R_OFF = ((IN_BYTES + 127) / 128) * 128;
    static constexpr int F_OFF = R_OFF + R_BYTES;
    static constexpr int STAGE_BYTES = ((F_OFF + F_BYTES + 127) / 128) * 128;
    static constexpr int XR_BYTES = ((n * n * C * (int)sizeof(TC) + 127) / 128) * 128;
    static constexpr int STAGES_ = (220 * 1024 - 2 * XR_BYTES) / STAGE_BYTES;
    static constexpr int STAGES = STAGES_ < 8 ? STAGES_ : 8;
    static constexpr size_t SMEM = (size_t)STAGES * STAGE_BYTES + 2 * XR_BYTES;
};

__device__ __forceinline__ void red_add(double* p, double v) { atomicAdd(p, v); }   // result unused -> RED.E.ADD.F64
__device__ __forceinline__ void red_add(float* p, float v) { atomicAdd(p, v); }

// the outputs (K v)_row(l), l < NJ, of half JH, from a whole line v
template <int P, int JH, typename TC>
__device__ __forceinline__ void eo_apply(const EoTab<TC>& tb, const TC (&v)[P + 1], TC (&out)[RowSet<P, JH>::NJ]) {
    using RS = RowSet<P, JH>;
    constexpr int H = RS::H, MID = RS::MID;
    TC ve[H], vo[H];
#pragma unroll
    for (int b = 0; b < H; ++b) { ve[b] = v[b] + v[P - b]; vo[b] = v[b] - v[P - b]; }
    const TC vm = v[MID];
#pragma unroll
    for (int p = 0; p < RS::NPAIR; ++p) {
        const int q = RS::Q0 + p;
        TC e = tb.Am[q] * vm, o = tb.B[q][0] * vo[0];
#pragma unroll
        for (int b = 0; b < H; ++b) e = fma(tb.A[q][b], ve[b], e);
#pragma unroll
        for (int b = 1; b < H; ++b) o = fma(tb.B[q][b], vo[b], o);
        out[2 * p] = e + o;
        out[2 * p + 1] = e - o;
    }
    if (RS::HASMID) {
        TC mm = tb.Mid[H] * vm;
#pragma unroll
        for (int b = 0; b < H; ++b) mm = fma(tb.Mid[b], ve[b], mm);
        out[RS::NJ - 1] = mm;
    }
}

template <int P, int CC, int MODE, bool HASPH, bool MASSIN, int JH>
struct XyzConsumer {
    using Cfg = XyzCfg<P, CC, MODE>;
    using RS = RowSet<P, JH>;
    using TI = typename Cfg::TI;
    using TC = typename Cfg::TC;
    using TO = typename ModeT<MODE>::TO;
    static constexpr int n = Cfg::n, C = Cfg::C, STAGES = Cfg::STAGES, NJ = RS::NJ;

    TC acc[n][NJ];              // z-accumulators of the current cell: acc[k][l], plane k, footprint row row(l), x-position a
    TC wxy[NJ];                 // W_x[a] W_y[row(l)]
    TC WXa, WYa;                // W_x[a] (YZ-phase), W_y[q] (X-phase: q is the row)
    double cin, cR, sg, mxa;
    double pXr, pXi;            // Bloch phase of the x-wrap at this thread's x-position ((1, 0) if it does not wrap)
    TO* outcol;                 // out + column offset + (line ey*P, x-position a)
    long long LS, PS;           // elements of `out` between consecutive y-lines / planes
    int a, col, s_spin, ri, g0;
    int rowoff, faceoff, voff, vstr;
    bool valid, emit_ok, own_a, xph, yph, ywrap;

    __device__ __forceinline__ void init(const XyzConst<TC>& sc, const MarchArgs& ar, int q, int col_, int ex, int ey, int chunk,
                                         int g0_, bool xwrap, bool ywrap_) {
        valid = q < n;
        a = valid ? q : P; col = col_; g0 = g0_; ywrap = ywrap_;
        xph = xwrap && ar.phd[0]; yph = ywrap && ar.phd[1];
        s_spin = col / (C / 2); ri = col & 1;
        sg = ((ri == 0) != (s_spin == 0)) ? -1.0 : 1.0;
        const int vl = (col % (C / 2)) >> 1;
        const int v = chunk * Cfg::NV + vl;
        const bool vok = v < ar.nvec;
        emit_ok = valid && vok;
        own_a = a < P;
        WXa = sc.WX[a]; WYa = sc.WY[a]; mxa = sc.M1X[a];
#pragma unroll
        for (int l = 0; l < NJ; ++l) wxy[l] = MODE == M_F64 ? (TC)0 : WXa * sc.WY[RS::row(l)];
        cin = (vok && ar.cin) ? __ldg(ar.cin + v) : 0.0;
        cR = (vok && ar.cR && ar.useR) ? __ldg(ar.cR + v) : 0.0;
        rowoff = a * P * C + col; faceoff = (n * P + a) * C + col;            // X-phase: row q of the plane
        voff = (own_a ? a * C : n * P * C) + col; vstr = own_a ? P * C : C;   // YZ-phase: y-line at x-position a
        pXr = 1.0; pXi = 0.0;
        int gx = ex * P + a;
        if (gx == ar.n1[0]) { gx = 0; if (HASPH && ar.phd[0]) { pXr = ar.ph_re[0]; pXi = ar.ph_im[0]; } }
        LS = (long long)ar.n1[0] * 4 * ar.ld_out;
        PS = (long long)ar.n1[1] * LS;
        outcol = reinterpret_cast<TO*>(ar.out) + ((long long)s_spin * ar.ld_out + (vok ? v : 0)) * 2 + ri +
                 (long long)ey * P * LS + (long long)gx * 4 * ar.ld_out;
#pragma unroll
        for (int k = 0; k < n; ++k)
#pragma unroll
            for (int l = 0; l < NJ; ++l) acc[k][l] = (TC)0;
    }

    // emit planes [0, nk) of the accumulators to global planes gzb + k (S3: one RED.ADD per node and column)
    __device__ __forceinline__ void emit(const XyzConst<TC>& sc, const MarchArgs& ar, int gzb, int nk) {
#pragma unroll
        for (int k = 0; k < n; ++k) {
            if (k < nk) {
                int gz = gzb + k; const bool wz = gz == ar.n1[2]; if (wz) gz = 0;
                if (HASPH) {
                    // conj(phase) of wrapped outputs: the x-wrap is per thread, the y-wrap is row P, the z-wrap is this plane
                    const bool zp = wz && ar.phd[2];
                    if (xph | yph | zp) {                                // CTA-uniform
                        double pr = pXr, pi = pXi;
                        if (zp) { const double t0 = pr * ar.ph_re[2] - pi * ar.ph_im[2]; pi = pr * ar.ph_im[2] + pi * ar.ph_re[2]; pr = t0; }
                        double qr = pr, qi = pi;                         // row P when it wraps in y
                        if (yph) { const double t0 = pr * ar.ph_re[1] - pi * ar.ph_im[1]; qi = pr * ar.ph_im[1] + pi * ar.ph_re[1]; qr = t0; }
                        if (ri) { pi = -pi; qi = -qi; }                  // re' = re pr + im pi ; im' = im pr - re pi
#pragma unroll
                        for (int l = 0; l < NJ; ++l) {
                            const TC val = acc[k][l];
                            const TC other = __shfl_xor_sync(0xffffffffu, val, 1);
                            const double cr = RS::row(l) == P ? qr : pr, ci = RS::row(l) == P ? qi : pi;
                            acc[k][l] = (TC)fma((double)other, ci, (double)val * cr);
                        }
                    }
                }
                if (emit_ok) {
                    TO* pk = outcol + gz * PS;
#pragma unroll
                    for (int l = 0; l < NJ; ++l) {
                        // row P of the last cell row is the global line y = 0 (outcol sits at line ey*P = N1y - P)
                        TO* dst = (RS::row(l) == P && ywrap) ? pk - (long long)(ar.n1[1] - P) * LS : pk + RS::row(l) * LS;
                        if (MODE == M_F32P) red_add(dst, (TO)(sc.cH * (double)acc[k][l]));
                        else red_add(dst, (TO)acc[k][l]);
                    }
                }
            }
        }
    }

    template <int K>
    __device__ __forceinline__ void add_plane(TC wzc, const TC (&ip)[NJ], const TC (&s5)[NJ]) {
        if constexpr (K < n) {
#pragma unroll
            for (int l = 0; l < NJ; ++l) {
                if constexpr (MODE == M_F64) acc[K][l] += ip[l];          // ip already holds w_z ip + S5
                else acc[K][l] += fma(wzc, ip[l], s5[l]);
            }
        }
    }

    // X-phase of plane t: this thread's row q = a of the plane, outputs at the x-positions row(l) of its half
    __device__ __forceinline__ void xphase(const XyzConst<TC>& sc, const MarchArgs& ar, unsigned char* smem, TC* XRbase, int t) {
        TI* IN = reinterpret_cast<TI*>(smem + (size_t)(t % STAGES) * Cfg::STAGE_BYTES);
        TC* XR = XRbase + (size_t)(t & 1) * (Cfg::XR_BYTES / sizeof(TC));
        if (HASPH) {
            // Bloch phase on wrapped entries of the plane (x: entry P of every row; y: the whole row P; z: the whole wrapped
            // plane), fixed up in place by half 0 before any row or line of the plane is read (boundary CTAs only)
            const bool wz = ar.phd[2] && (g0 + t) == ar.n1[2];
            if (xph | yph | wz) {                                        // CTA-uniform
                const bool wyy = yph && a == P;
                double br = 1.0, bi = 0.0;                               // phase of the whole row (y- and z-wrap)
                if (wyy) { br = ar.ph_re[1]; bi = ar.ph_im[1]; }
                if (wz) { const double t0 = br * ar.ph_re[2] - bi * ar.ph_im[2]; bi = br * ar.ph_im[2] + bi * ar.ph_re[2]; br = t0; }
                const double s1 = ri ? 1.0 : -1.0;                       // re' = re pr - im pi ; im' = im pr + re pi
                if (JH == 0) {
#pragma unroll
                    for (int i = 0; i < n; ++i) {
                        double pr = br, pi = bi;
                        if (i == P && xph) { const double t0 = pr * ar.ph_re[0] - pi * ar.ph_im[0]; pi = pr * ar.ph_im[0] + pi * ar.ph_re[0]; pr = t0; }
                        const int o = i < P ? rowoff + i * C : faceoff;
                        const TI val = IN[o];
                        const TI other = IN[o + ((col ^ 1) - col)];      // the partner lane rewrites it: read before the sync
                        __syncwarp();
                        if (((wyy | wz) || (i == P && xph)) && valid) IN[o] = (TI)fma((double)other, s1 * pi, (double)val * pr);
                    }
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // these stage bytes are later rewritten by TMA
                }
                asm volatile("bar.sync 1, %0;" ::"r"(Cfg::NCW * 32) : "memory");    // consumer warps only
            }
        }
        TI rw[n];
#pragma unroll
        for (int i = 0; i < P; ++i) rw[i] = IN[rowoff + i * C];
        rw[P] = IN[faceoff];
        TC rv[n], sx[NJ];
#pragma unroll
        for (int i = 0; i < n; ++i) rv[i] = (MODE == M_F32P) ? (TC)(rw[i] * (TI)sc.in_scale) : (TC)rw[i];
        eo_apply<P, JH, TC>(sc.X, rv, sx);
        if (valid) {
#pragma unroll
            for (int l = 0; l < NJ; ++l) XR[(a * n + RS::row(l)) * C + col] = WYa * sx[l];
        }
    }

    // YZ-phase of plane t.  c = its local index in the current cell (upper role); lower: it is also plane P of the
    // previous cell; upper: it belongs to a cell of this segment (false only for the segment's last plane).
    // next: the X-phase of plane t + 1 is computed first.
    __device__ __forceinline__ void step(const XyzConst<TC>& sc, const MarchArgs& ar, unsigned char* smem, TC* XRbase,
                                         uint64_t* full_bar, uint64_t* empty_bar, int t, int c, bool lower, bool upper, bool next) {
        const int s = t % STAGES;
        TI* IN = reinterpret_cast<TI*>(smem + (size_t)s * Cfg::STAGE_BYTES);
        const double* Rs = reinterpret_cast<const double*>(smem + (size_t)s * Cfg::STAGE_BYTES + Cfg::R_OFF);
        const double* Fs = reinterpret_cast<const double*>(smem + (size_t)s * Cfg::STAGE_BYTES + Cfg::F_OFF);
        const TC* XR = XRbase + (size_t)(t & 1) * (Cfg::XR_BYTES / sizeof(TC));
        if (next) {
            // X-phase of the next plane first: XR[(t+1)&1] was last read in the YZ-phase of plane t-1, which every warp
            // finished before the barrier that ended the previous step.  (Measured on configs[3]: this order with one
            // bar.sync per plane, 8.9 ms; X-phase between the loads and the arithmetic of plane t, 9.1 ms; an mbarrier
            // full/empty handshake on XR instead of the barrier, 9.3-9.4 ms.)
            mbar_wait(&full_bar[(t + 1) % STAGES], ((t + 1) / STAGES) & 1);
            xphase(sc, ar, smem, XRbase, t + 1);
        }
        TI vin[n];
        TC v[n], ip[NJ];
#pragma unroll
        for (int b = 0; b < n; ++b) vin[b] = IN[voff + b * vstr];
#pragma unroll
        for (int l = 0; l < NJ; ++l) ip[l] = XR[(RS::row(l) * n + a) * C + col];
#pragma unroll
        for (int b = 0; b < n; ++b) v[b] = (MODE == M_F32P) ? (TC)(vin[b] * (TI)sc.in_scale) : (TC)vin[b];
        {
            TC sy[NJ];
            eo_apply<P, JH, TC>(sc.Y, v, sy);
#pragma unroll
            for (int l = 0; l < NJ; ++l) ip[l] = fma(WXa, sy[l], ip[l]);
        }
        TC zr[NJ];
#pragma unroll
        for (int l = 0; l < NJ; ++l) {
            // FP64: the product W_x[a] W_y[row] is not kept per thread (NJ double registers under the 168-register cap); the
            // weight of the row comes from the constant bank and the association keeps the compiler from hoisting it back
            if constexpr (MODE == M_F64) zr[l] = WXa * (sc.WY[RS::row(l)] * v[RS::row(l)]);
            else zr[l] = wxy[l] * v[RS::row(l)];
        }
        if (lower) {
#pragma unroll
            for (int k = 0; k < n; ++k) {
                const TC kz = sc.KZ[k][P];
#pragma unroll
                for (int l = 0; l < NJ; ++l) acc[k][l] = fma(kz, zr[l], acc[k][l]);
            }
#pragma unroll
            for (int l = 0; l < NJ; ++l) acc[P][l] = fma(sc.WZ[P], ip[l], acc[P][l]);
            // the previous cell is complete: emit its planes 0..P-1, carry its top plane over
            emit(sc, ar, g0 + t - P, P);
#pragma unroll
            for (int l = 0; l < NJ; ++l) acc[0][l] = acc[P][l];
#pragma unroll
            for (int k = 1; k < n; ++k)
#pragma unroll
                for (int l = 0; l < NJ; ++l) acc[k][l] = (TC)0;
        }
        if (upper) {
            // z-push with the runtime cell-local index c: column c of KZ fetched from the constant bank
#pragma unroll
            for (int k = 0; k < n; ++k) {
                const TC kz = sc.KZ[k][c];
#pragma unroll
                for (int l = 0; l < NJ; ++l) acc[k][l] = fma(kz, zr[l], acc[k][l]);
            }
            // FP64: S5 is folded into the in-plane part as it is formed (ip <- w_z ip + S5), so no second array of NJ values is live
            const TC wzc = sc.WZ[c];
            TC s5[NJ];
#pragma unroll
            for (int l = 0; l < NJ; ++l) s5[l] = (TC)0;
            if constexpr (MODE == M_F64) {
                if (!own_a) {
#pragma unroll
                    for (int l = 0; l < NJ; ++l) ip[l] = wzc * ip[l];
                }
            }
            if (own_a) {
                // S5 on the owned nodes of this plane (rows < P at x-position a < P): eq. 12 spin blocks, in-term, R-term
                const int nb = a * C + col;
                const double mzx = MASSIN ? sc.M1Z[c] * mxa : 1.0;
                [[maybe_unused]] TO* p5 = outcol + (long long)(g0 + t) * PS;
#pragma unroll
                for (int l = 0; l < NJ; ++l) {
                    const int j = RS::row(l);
                    if (j < P) {
                        // (B_x -+ i B_y) u_other: B_x * (other spin, same part) + sg * B_y * (other spin, other part)
                        const int o = j * P * C + nb;
                        if constexpr (MODE == M_F32S) {
                            // FP32-stored multivectors (only R and Lambda_k stay FP64): FP32 pointwise terms on
                            // the FP32 copy of the fields; the R-term is formed in FP64 and rounded once
                            const float4 f = *reinterpret_cast<const float4*>(reinterpret_cast<const float*>(Fs) + (j * P + a) * 4);
                            const float in_f = vin[j];
                            const float os = IN[o + ((col ^ (C / 2)) - col)], of = IN[o + ((col ^ (C / 2 + 1)) - col)];
                            const float pot = fmaf(s_spin ? f.y : f.x, in_f, fmaf(f.z, os, ((float)sg * f.w) * of));
                            float val = fmaf((float)cin, in_f, (float)sc.cHp * pot);
                            if (ar.useR) val += (float)(cR * Rs[o]);
                            s5[l] = val;
                            continue;
                        }
                        const double in_own = (double)vin[j];
                        const double o_same = (double)IN[o + ((col ^ (C / 2)) - col)];
                        const double o_flip = (double)IN[o + ((col ^ (C / 2 + 1)) - col)];
                        const double diag = Fs[(j * P + a) * 4 + s_spin];
                        const double2 bxy = *reinterpret_cast<const double2*>(Fs + (j * P + a) * 4 + 2);
                        const double pot = fma(diag, in_own, fma(bxy.x, o_same, (sg * bxy.y) * o_flip));
                        double val = fma(cin, in_own, sc.cHp * pot);
                        if (MASSIN) val *= mzx * sc.M1Y[j];              // the residual S0: H X - M X Lambda carries m_I
                        if (ar.useR) val = fma(cR, Rs[o], val);
                        if (MODE == M_F32P) { if (emit_ok) red_add(p5 + (long long)j * LS, (TO)val); }
                        else if (MODE == M_F64) ip[l] = fma(wzc, ip[l], (TC)val);
                        else s5[l] = (TC)val;
                    } else if (MODE == M_F64) {
                        ip[l] = wzc * ip[l];
                    }
                }
            }
            switch (c) {
                case 0: add_plane<0>(wzc, ip, s5); break;
                case 1: add_plane<(1 < P ? 1 : n)>(wzc, ip, s5); break;
                case 2: add_plane<(2 < P ? 2 : n)>(wzc, ip, s5); break;
                case 3: add_plane<(3 < P ? 3 : n)>(wzc, ip, s5); break;
                case 4: add_plane<(4 < P ? 4 : n)>(wzc, ip, s5); break;
                case 5: add_plane<(5 < P ? 5 : n)>(wzc, ip, s5); break;
                case 6: add_plane<(6 < P ? 6 : n)>(wzc, ip, s5); break;
                default: add_plane<(7 < P ? 7 : n)>(wzc, ip, s5); break;
            }
        }
        __syncwarp();
        if ((threadIdx.x & 31) == 0) mbar_arrive(&empty_bar[s]);
        asm volatile("bar.sync 1, %0;" ::"r"(Cfg::NCW * 32) : "memory");      // consumer warps only: XR of plane t + 1 is complete
    }

    __device__ __forceinline__ void run(const XyzConst<TC>& sc, const MarchArgs& ar, unsigned char* smem, TC* XR, uint64_t* full_bar,
                                        uint64_t* empty_bar, int T) {
        mbar_wait(&full_bar[0], 0);
        xphase(sc, ar, smem, XR, 0);
        asm volatile("bar.sync 1, %0;" ::"r"(Cfg::NCW * 32) : "memory");
        int c = 0;
#pragma unroll 1
        for (int t = 0; t < T; ++t) {
            step(sc, ar, smem, XR, full_bar, empty_bar, t, c, c == 0 && t > 0, t < T - 1, t < T - 1);
            c = (c + 1 == P) ? 0 : c + 1;
        }
        emit(sc, ar, g0 + T - 1, 1);                                   // partial of the segment's top face
    }
};

template <int P, int CC, int MODE, bool HASPH, bool MASSIN>
__global__ void __launch_bounds__(XyzCfg<P, CC, MODE>::THREADS, 1)
cell_xyz_kernel(const __grid_constant__ XyzConst<typename ModeT<MODE>::TC> sc, const __grid_constant__ MarchArgs ar,
                const __grid_constant__ MarchMaps mp) {
    using Cfg = XyzCfg<P, CC, MODE>;
    using TC = typename Cfg::TC;
    constexpr int C = Cfg::C, STAGES = Cfg::STAGES;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t full_bar[STAGES], empty_bar[STAGES];
    TC* XR = reinterpret_cast<TC*>(smem + (size_t)STAGES * Cfg::STAGE_BYTES);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // blockIdx -> (ex fastest, ey, seg, chunk): neighbours in x/y run together, so shared faces hit in L2.
    // When a row of the CTA's columns is shorter than a 128-byte line (PAIR chunks share one), they run side by side.
    constexpr int ROWB = (C / 2) * (int)sizeof(typename Cfg::TI);
    constexpr int PAIR = ROWB >= 128 ? 1 : 128 / ROWB;
    int bid = blockIdx.x;
    const int cpair = bid % PAIR; bid /= PAIR;
    const int ex = bid % ar.nc[0]; bid /= ar.nc[0];
    const int ey = bid % ar.nc[1]; bid /= ar.nc[1];
    const int seg = bid % ar.nseg;
    const int chunk = PAIR * (bid / ar.nseg) + cpair;
    if (chunk >= ar.nchunks) return;              // chunk count not a multiple of PAIR: the last group is partly empty
    const int T = ar.cps * P + 1;                 // planes this CTA marches through
    const int g0 = seg * ar.cps * P;              // first global plane
    const bool xwrap = ex == ar.nc[0] - 1, ywrap = ey == ar.nc[1] - 1;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], Cfg::NCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == Cfg::NCW) {
        // ================================ producer ================================
        if (lane == 0) {
            const int col0 = chunk * (C / 2);                     // elements of the (node, spin) row
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
                constexpr int ESZ = (int)sizeof(typename Cfg::TI);
                if (!ywrap) {
                    tma_load_3d(st, &mp.main[0], col0, xr, line, &full_bar[s]);
                    tma_load_3d(st + Cfg::FACE_OFF, &mp.face[0], col0, xf, line, &full_bar[s]);
                } else {
                    tma_load_3d(st, &mp.main[1], col0, xr, line, &full_bar[s]);
                    tma_load_3d(st + P * P * C * ESZ, &mp.main[2], col0, xr, gz * ar.n1[1], &full_bar[s]);
                    tma_load_3d(st + Cfg::FACE_OFF, &mp.face[1], col0, xf, line, &full_bar[s]);
                    tma_load_3d(st + Cfg::FACE_OFF + P * C * ESZ, &mp.face[2], col0, xf, gz * ar.n1[1], &full_bar[s]);
                }
                if (owned) {
                    if (ar.useR) tma_load_3d(st + Cfg::R_OFF, &mp.R, col0, xr, line, &full_bar[s]);
                    tma_load_2d_hint(st + Cfg::F_OFF, &mp.F, 4 * ex * P, line, &full_bar[s], pol_last);
                }
            }
        }
        return;
    }

    // ================================ consumers ================================
    // warp w: half jh = w % 2 of the rows, indices q = (w / 2) * RPW + lane / C (the half-empty warps of C = 16 come last)
    // Role r of warp w (half jh = r % 2, index group r / 2).  Warps go to the four schedulers of the SM by w % 4 and the
    // half-0 warps carry one row more (NJ = 5 against 4 at p = 8), so the plain r = w would put every heavy warp on
    // schedulers 0 and 2.  Ten consumer warps (p = 8, C = 16; schedulers hold 3, 3, 2 + producer, 2 warps): heavy warps on the
    // two-warp schedulers.  Otherwise: swap the halves in every other group of four warps.
    int role = warp ^ ((warp >> 2) & 1);
    if (Cfg::NCW == 10) role = (int)((0x9562734081ull >> (4 * warp)) & 15);   // w: 0 1 2 3 4 5 6 7 8 9 -> r: 1 8 0 4 3 7 2 6 5 9
    const int q = (role >> 1) * Cfg::RPW + lane / C;
    if ((role & 1) == 0) {
        XyzConsumer<P, CC, MODE, HASPH, MASSIN, 0> cs;
        cs.init(sc, ar, q, lane % C, ex, ey, chunk, g0, xwrap, ywrap);
        cs.run(sc, ar, smem, XR, full_bar, empty_bar, T);
    } else {
        XyzConsumer<P, CC, MODE, HASPH, MASSIN, 1> cs;
        cs.init(sc, ar, q, lane % C, ex, ey, chunk, g0, xwrap, ywrap);
        cs.run(sc, ar, smem, XR, full_bar, empty_bar, T);
    }
}

// ---------------------------------------------------------------------------------------------
template <typename TC>
static void build_eo(EoTab<TC>& tb, const double (*K)[kMaxN], int P) {
    const int H = (P + 1) / 2, MID = P / 2;
    std::memset(&tb, 0, sizeof(tb));
    for (int j = 0; j < H; ++j) {
        for (int b = 0; b < H; ++b) {
            // impose exact centrosymmetry: average K[j][b] with K[P-j][P-b] (equal up to rounding of the GLL tables)
            const double kjb = 0.5 * (K[j][b] + K[P - j][P - b]), kjq = 0.5 * (K[j][P - b] + K[P - j][b]);
            tb.A[j][b] = (TC)(0.5 * (kjb + kjq));
            tb.B[j][b] = (TC)(0.5 * (kjb - kjq));
        }
        tb.Am[j] = (TC)(0.5 * (K[j][MID] + K[P - j][MID]));
    }
    for (int b = 0; b < H; ++b) tb.Mid[b] = (TC)(0.5 * (K[MID][b] + K[MID][P - b]));
    tb.Mid[H] = (TC)K[MID][MID];
}

// All scalings (1/2, Jacobian, D^-1 on the way in, M^-1 on the way out, the step coefficient) are folded into the
// per-launch 1-D tables, so the inner loops are bare FMAs with constant-bank operands.
template <typename TC>
static void build_const(const chfsi_mesh* m, const CellArgs& a, bool fold_cH, XyzConst<TC>& sc) {
    const MeshConst& mc = m->mc;
    const int n = mc.n, P = mc.p;
    const bool sin_ = (a.flags & kScaleIn) != 0, sout_ = (a.flags & kSoutInvM) != 0;
    std::memset(&sc, 0, sizeof(sc));
    const double isc = a.in_scale > 0.0 ? a.in_scale : 1.0;        // used by the FP32 product only
    sc.cH = a.cH / isc;
    sc.in_scale = isc;
    // coefficient of the potential term: cH * s_out * (u / in) with u = m w.  In the Z-form (w = in / m, no s_out) and in
    // the M^-1 H form (w = in, s_out = 1/m) that product is cH at every node; in the residual form (w = in, no s_out) it
    // is cH m_I, which the MASSIN kernel applies together with the mass of the in-term.
    sc.cHp = a.cH;
    const double ch = fold_cH ? a.cH : 1.0;
    double K[3][kMaxN][kMaxN];
    for (int d = 0; d < 3; ++d) {
        TC* W = d == 0 ? sc.WX : d == 1 ? sc.WY : sc.WZ;
        double* M1 = d == 0 ? sc.M1X : d == 1 ? sc.M1Y : sc.M1Z;
        for (int i = 0; i < n; ++i) {
            const double si = sin_ ? mc.im1[d][i] : 1.0, so = sout_ ? mc.im1[d][i] : 1.0;
            for (int b = 0; b < n; ++b) {
                const double sb = sin_ ? mc.im1[d][b] : 1.0;
                K[d][i][b] = (d == 0 ? ch : 1.0) * so * mc.Kd[d][i][b] * sb;
            }
            // the step coefficient rides on the x-direction factors: on K_x for the x-part, and on W_x, which multiplies
            // the y- and z-parts (and never meets K_x)
            W[i] = (TC)((d == 0 ? ch : 1.0) * mc.w[i] * so * si);
            M1[i] = mc.m1[d][i];
        }
    }
    build_eo(sc.X, K[0], P);
    build_eo(sc.Y, K[1], P);
    for (int k = 0; k < n; ++k)
        for (int c = 0; c < n; ++c) sc.KZ[k][c] = (TC)K[2][k][c];
}

static std::once_flag g_attr_once[4][3][4][32];   // [p/2 - 1][mode][phase, massin][device]

template <int P, int CC, int MODE>
static cudaError_t launch_xyz_t(const chfsi_mesh* m, const CellArgs& a, cudaStream_t st) {
    using Cfg = XyzCfg<P, CC, MODE>;
    using TC = typename Cfg::TC;
    using TI = typename Cfg::TI;
    XyzConst<TC> sc;
    build_const<TC>(m, a, MODE != M_F32P, sc);
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
    constexpr bool f32in = sizeof(TI) == 4;
    const int nl[3] = {P + 1, P, 1};
    for (int i = 0; i < 3; ++i)
        if (!make_map3(&mp.main[i], m, a.in, a.ld_in, a.nvec, BC, 2 * P, nl[i], f32in) ||
            !make_map3(&mp.face[i], m, a.in, a.ld_in, a.nvec, BC, 2, nl[i], f32in))
            return cudaErrorInvalidValue;
    if (!make_map3(&mp.R, m, ar.useR ? a.R : a.in, ar.useR ? a.ld_R : a.ld_in, a.nvec, BC, 2 * P, P, ar.useR ? false : f32in) ||
        !make_mapF(&mp.F, m, P, MODE == M_F32S))
        return cudaErrorInvalidValue;
    const bool ph = m->mc.has_phase != 0;
    // the mass of the in-term and of the potential term (residual form) needs the flags kMassIn alone
    const bool massin = (a.flags & kMassIn) != 0;
    if (massin && (a.flags & (kScaleIn | kSoutInvM))) return cudaErrorInvalidValue;
    constexpr bool MI = MODE == M_F64;            // the residual form is only ever run in FP64
    if (massin && !MI) return cudaErrorInvalidValue;
    auto kern = ph ? (massin ? cell_xyz_kernel<P, CC, MODE, true, MI> : cell_xyz_kernel<P, CC, MODE, true, false>)
                   : (massin ? cell_xyz_kernel<P, CC, MODE, false, MI> : cell_xyz_kernel<P, CC, MODE, false, false>);
    cudaError_t attr_err = cudaSuccess;
    std::call_once(g_attr_once[P / 2 - 1][MODE][(ph ? 2 : 0) + (massin ? 1 : 0)][m->device & 31], [&] {
        attr_err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
    });
    if (attr_err != cudaSuccess) return attr_err;
    constexpr int ROWB = (CC / 2) * (int)sizeof(TI);
    constexpr int PAIR = ROWB >= 128 ? 1 : 128 / ROWB;
    const long long grid = (long long)ar.nc[0] * ar.nc[1] * nseg * PAIR * ((ar.nchunks + PAIR - 1) / PAIR);
    kern<<<(unsigned)grid, Cfg::THREADS, Cfg::SMEM, st>>>(sc, ar, mp);
    return cudaGetLastError();
}

bool xyz_supported(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a) {
    if (prec != CHFSI_FP64 && prec != CHFSI_FP32 && prec != CHFSI_FP32_STORED) return false;
    if ((prec == CHFSI_FP32_STORED) != (a.store_f32 != 0)) return false;
    if (m->p != 2 && m->p != 4 && m->p != 6 && m->p != 8) return false;
    if (m->dF == nullptr) return false;
    if (prec != CHFSI_FP64 && (a.flags & kMassIn)) return false;      // the residual S0 is always FP64
    // TMA needs 16-byte aligned bases and row pitches (always true for complex128 rows; an even leading dimension for
    // complex64) and 32-bit row coordinates
    if (2 * m->nnodes >= (1ll << 31)) return false;
    if (a.store_f32 && ((a.ld_in & 1) || (a.ld_out & 1))) return false;
    if (((uintptr_t)a.in & 15) || ((uintptr_t)a.out & 15) || (a.R && ((uintptr_t)a.R & 15))) return false;
    return get_encode() != nullptr;
}

cudaError_t launch_cell_xyz(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t st) {
    if (prec == CHFSI_FP32_STORED) {
        switch (m->p) {
            case 2: return launch_xyz_t<2, 32, M_F32S>(m, a, st);
            case 4: return launch_xyz_t<4, 32, M_F32S>(m, a, st);
            case 6: return launch_xyz_t<6, 32, M_F32S>(m, a, st);
            case 8: return launch_xyz_t<8, 32, M_F32S>(m, a, st);
            default: return cudaErrorInvalidValue;
        }
    }
    if (prec == CHFSI_FP32) {
        switch (m->p) {
            case 2: return launch_xyz_t<2, 32, M_F32P>(m, a, st);
            case 4: return launch_xyz_t<4, 32, M_F32P>(m, a, st);
            case 6: return launch_xyz_t<6, 32, M_F32P>(m, a, st);
            case 8: return launch_xyz_t<8, 32, M_F32P>(m, a, st);
            default: return cudaErrorInvalidValue;
        }
    }
    switch (m->p) {
        case 2: return launch_xyz_t<2, 32, M_F64>(m, a, st);
        case 4: return launch_xyz_t<4, 32, M_F64>(m, a, st);
        case 6: return launch_xyz_t<6, 32, M_F64>(m, a, st);
        case 8: return launch_xyz_t<8, 16, M_F64>(m, a, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace chfsi
