// sm_100a kernels of libchfsi: cell gather / sum-factorised Laplacian / fused pointwise update with
// in-place L2 reductions (S1-S3, S5, S6 of DESIGN.md), nonlocal projector kernels (S4), and the
// pointwise recover/scale kernel (S7).
#include <cstdlib>

#include "chfsi_internal.h"

namespace chfsi {

// ---------------------------------------------------------------------------------------------
// helpers
template <typename TT> struct KSel;
template <> struct KSel<double> {
    static __device__ __forceinline__ double K(const MeshConst& mc, int d, int i, int a) { return mc.Kd[d][i][a]; }
    static __device__ __forceinline__ double w(const MeshConst& mc, int a) { return mc.w[a]; }
};
template <> struct KSel<float> {
    static __device__ __forceinline__ float K(const MeshConst& mc, int d, int i, int a) { return mc.Kf[d][i][a]; }
    static __device__ __forceinline__ float w(const MeshConst& mc, int a) { return mc.wf[a]; }
};

__device__ __forceinline__ void red_add(double* p, double v) { atomicAdd(p, v); }  // result unused -> RED.E.ADD.F64

// ---------------------------------------------------------------------------------------------
// Cell kernel.  One CTA = one FE cell x NV complex vectors (C = 4 NV real batch columns: re/im of both
// spin components, which the spin-diagonal real Laplacian treats alike -- north_star kernel (1)/(2)).
//   S1 gather   : W^(e) = R^(e) (s_in * in)           (PAPER.md:204 stage (i); Bloch phase on wrapped nodes)
//   S2 Laplacian: T^(e) = 1/2 K_e W^(e) by three 1-D contractions
//                 pass 1: each thread owns one xy-plane of one column, x- and y-contractions in registers
//                 pass 2: each thread owns z-lines, z-contraction in registers, straight into the epilogue
//   S3 assembly : out[I] += conj(phase) * cH * s_out * T^(e)   (RED.ADD.F64 at L2; PAPER.md:204 stage (iii))
//   S5 pointwise: on the nodes the cell owns (local index < p in every direction) the 2x2 spin
//                 potential of eq. 12, the in-term and the R-term of eq. 11 are added in the same pass.
// Thread t: column col = t % C, group grp = t / C, G = n groups.
template <int P, int NV, typename TT>
__global__ void __launch_bounds__((P + 1) * 4 * NV)
cell_kernel(const __grid_constant__ MeshConst mc, const __grid_constant__ CellArgs ar) {
    constexpr int n = P + 1, n3 = n * n * n, C = 4 * NV, G = n;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TT* W = reinterpret_cast<TT*>(smem_raw);
    TT* T2 = W + n3 * C;

    const int tid = threadIdx.x;
    const int col = tid % C, grp = tid / C;
    const int cell = blockIdx.x % mc.ncells, chunk = blockIdx.x / mc.ncells;
    const int ex = cell % mc.nc[0], ey = (cell / mc.nc[0]) % mc.nc[1], ez = cell / (mc.nc[0] * mc.nc[1]);
    const int s = col / (2 * NV), vl = (col % (2 * NV)) >> 1, ri = col & 1;
    const int v = chunk * NV + vl;
    const bool vok = v < ar.nvec;
    const int flags = ar.flags;
    const bool hasph = mc.has_phase != 0;
    const double isc = ar.in_scale > 0.0 ? ar.in_scale : 1.0;

    // ---- S1 gather
    {
        const double* __restrict__ src = ar.in + ((long long)s * ar.ld_in + v) * 2 + ri;
        for (int l = grp; l < n3; l += G) {
            const int a = l % n, b = (l / n) % n, c = l / (n * n);
            int gx = ex * P + a, gy = ey * P + b, gz = ez * P + c;
            const bool wx = gx == mc.n1[0], wy = gy == mc.n1[1], wz = gz == mc.n1[2];
            gx = wx ? 0 : gx; gy = wy ? 0 : gy; gz = wz ? 0 : gz;
            const long long I = ((long long)gz * mc.n1[1] + gy) * mc.n1[0] + gx;
            double val = vok ? __ldg(src + I * 4 * ar.ld_in) : 0.0;
            if (hasph) {
                const double other = __shfl_xor_sync(__activemask(), val, 1);
                if (wx | wy | wz) {
                    double pr = 1.0, pi = 0.0;
                    if (wx) { pr = mc.ph_re[0]; pi = mc.ph_im[0]; }
                    if (wy) { const double t = pr * mc.ph_re[1] - pi * mc.ph_im[1]; pi = pr * mc.ph_im[1] + pi * mc.ph_re[1]; pr = t; }
                    if (wz) { const double t = pr * mc.ph_re[2] - pi * mc.ph_im[2]; pi = pr * mc.ph_im[2] + pi * mc.ph_re[2]; pr = t; }
                    // (re + i im)(pr + i pi): re' = re pr - im pi ; im' = re pi + im pr
                    val = ri == 0 ? val * pr - other * pi : other * pi + val * pr;
                }
            }
            if (flags & kScaleIn) val *= mc.im1[0][a] * mc.im1[1][b] * mc.im1[2][c];
            if (sizeof(TT) == 4) val *= isc;                         // keep Z_k / s_k inside the FP32 range
            W[l * C + col] = (TT)val;
        }
    }
    __syncthreads();

    // ---- S2 pass 1: xy-plane c = grp; T2[c][j][i] = w_c ( w_j (Kx W)_i + w_i (Ky W)_j )
    for (int c = grp; c < n; c += G) {
        TT o[n][n];
#pragma unroll
        for (int j = 0; j < n; ++j)
#pragma unroll
            for (int i = 0; i < n; ++i) o[j][i] = (TT)0;
#pragma unroll
        for (int b = 0; b < n; ++b) {
            TT in[n];
#pragma unroll
            for (int a = 0; a < n; ++a) in[a] = W[((c * n + b) * n + a) * C + col];
            const TT wb = KSel<TT>::w(mc, b);
#pragma unroll
            for (int i = 0; i < n; ++i) {
                TT sx = (TT)0;
#pragma unroll
                for (int a = 0; a < n; ++a) sx = fma(KSel<TT>::K(mc, 0, i, a), in[a], sx);
                o[b][i] = fma(wb, sx, o[b][i]);
            }
#pragma unroll
            for (int a = 0; a < n; ++a) {
                const TT t = KSel<TT>::w(mc, a) * in[a];
#pragma unroll
                for (int j = 0; j < n; ++j) o[j][a] = fma(KSel<TT>::K(mc, 1, j, b), t, o[j][a]);
            }
        }
        const TT wc = KSel<TT>::w(mc, c);
#pragma unroll
        for (int j = 0; j < n; ++j)
#pragma unroll
            for (int i = 0; i < n; ++i) T2[((c * n + j) * n + i) * C + col] = wc * o[j][i];
    }
    __syncthreads();

    // ---- S2 pass 2 + S3/S5 epilogue: z-lines (b,a)
    const double cin = (vok && ar.cin) ? __ldg(ar.cin + v) : 0.0;
    const double cR = (vok && ar.cR) ? __ldg(ar.cR + v) : 0.0;
    const bool useR = ar.R != nullptr && ar.cR != nullptr;
    for (int li = grp; li < n * n; li += G) {
        const int a = li % n, b = li / n;
        TT in[n], t[n];
#pragma unroll
        for (int c = 0; c < n; ++c) {
            in[c] = W[((c * n + b) * n + a) * C + col];
            t[c] = T2[((c * n + b) * n + a) * C + col];
        }
        const TT wab = KSel<TT>::w(mc, a) * KSel<TT>::w(mc, b);
#pragma unroll
        for (int k = 0; k < n; ++k) {
            TT sz = (TT)0;
#pragma unroll
            for (int c = 0; c < n; ++c) sz = fma(KSel<TT>::K(mc, 2, k, c), in[c], sz);
            t[k] = fma(wab, sz, t[k]);
        }
        int gx = ex * P + a, gy = ey * P + b;
        const bool wx = gx == mc.n1[0], wy = gy == mc.n1[1];
        gx = wx ? 0 : gx; gy = wy ? 0 : gy;
        const double mab = mc.m1[0][a] * mc.m1[1][b];
        const double imab = mc.im1[0][a] * mc.im1[1][b];
#pragma unroll
        for (int k = 0; k < n; ++k) {
            int gz = ez * P + k;
            const bool wz = gz == mc.n1[2];
            gz = wz ? 0 : gz;
            const long long I = ((long long)gz * mc.n1[1] + gy) * mc.n1[0] + gx;
            const double mI = mab * mc.m1[2][k];
            const double imI = imab * mc.im1[2][k];
            const double sout = (flags & kSoutInvM) ? imI : 1.0;
            double val = (sizeof(TT) == 4 ? ar.cH / isc : ar.cH) * sout * (double)t[k];
            if (hasph) {
                const double other = __shfl_xor_sync(__activemask(), val, 1);
                if (wx | wy | wz) {
                    double pr = 1.0, pi = 0.0;
                    if (wx) { pr = mc.ph_re[0]; pi = mc.ph_im[0]; }
                    if (wy) { const double tt = pr * mc.ph_re[1] - pi * mc.ph_im[1]; pi = pr * mc.ph_im[1] + pi * mc.ph_re[1]; pr = tt; }
                    if (wz) { const double tt = pr * mc.ph_re[2] - pi * mc.ph_im[2]; pi = pr * mc.ph_im[2] + pi * mc.ph_re[2]; pr = tt; }
                    // multiply by conj(phase): re' = re pr + im pi ; im' = im pr - re pi
                    val = ri == 0 ? val * pr + other * pi : val * pr - other * pi;
                }
            }
            if (a < P && b < P && k < P) {   // node owned by this cell: pointwise terms (never wrapped)
                const int l = (k * n + b) * n + a;
                // u = m_I * w for both spins / both parts of this vector.  FP64: recovered from the tile
                // (one extra rounding); FP32: re-read in FP64 so the recurrence terms stay exact FP64.
                double u_own, u_oth_re, u_oth_im, in_own;
                const int ocol = col ^ (2 * NV);            // same vector, other spin
                if (sizeof(TT) == 8) {
                    const double f = (flags & kScaleIn) ? mI : 1.0;      // in = w * f
                    in_own = (double)in[k] * f;
                    const double o_same = (double)W[l * C + ocol] * f;   // other spin, same part
                    const double o_flip = (double)W[l * C + (ocol ^ 1)] * f;
                    u_oth_re = ri == 0 ? o_same : o_flip;
                    u_oth_im = ri == 0 ? o_flip : o_same;
                } else {
                    const double* base = ar.in + I * 4 * ar.ld_in;
                    in_own = vok ? __ldg(base + ((long long)s * ar.ld_in + v) * 2 + ri) : 0.0;
                    const double2 oth = vok ? __ldg(reinterpret_cast<const double2*>(base + ((long long)(s ^ 1) * ar.ld_in + v) * 2))
                                            : make_double2(0.0, 0.0);
                    u_oth_re = oth.x; u_oth_im = oth.y;
                }
                const double fu = (flags & kScaleIn) ? 1.0 : mI;         // u = m w: Z-form u = in, else m * in
                u_own = in_own * fu;
                u_oth_re *= fu; u_oth_im *= fu;
                const double Vn = __ldg(mc.V + I), Bxn = __ldg(mc.Bx + I), Byn = __ldg(mc.By + I), Bzn = __ldg(mc.Bz + I);
                // eq. 12 spin blocks, pointwise: up: (V+Bz) u_up + (Bx - i By) u_dn ; dn: (Bx + i By) u_up + (V - Bz) u_dn
                const double diag = s == 0 ? Vn + Bzn : Vn - Bzn;
                const double sy = s == 0 ? -Byn : Byn;                   // off-diagonal = Bx + i sy
                // (Bx + i sy)(re + i im) = (Bx re - sy im) + i (Bx im + sy re)
                const double offd = ri == 0 ? Bxn * u_oth_re - sy * u_oth_im : Bxn * u_oth_im + sy * u_oth_re;
                val += ar.cH * sout * (diag * u_own + offd);
                val += cin * ((flags & kMassIn) ? mI : 1.0) * in_own;
                if (useR && vok) val += cR * __ldg(ar.R + ((2 * I + s) * ar.ld_R + v) * 2 + ri);
            }
            if (vok) red_add(ar.out + ((2 * I + s) * ar.ld_out + v) * 2 + ri, val);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// S4 nonlocal term (PAPER.md:204 stage (iv)): three small kernels per H application.
//   proj : C_a[2 beta + s][v] += sum_{I in slice} conj(P_a[I,beta]) u_{I,s,v}      (skinny GEMM, RED into C)
//   gmat : G_a = D_a C_a                                                            ((2 nproj)^2 per atom)
//   back : out_{I,s,v} += cH * f_I * sum_beta P_a[I,beta] G_a[2 beta + s][v]        (RED into out)
// A slice is kSlice support nodes, fully unrolled so that all its loads are in flight at once; one CTA =
// one slice x 128 (spin, vector) columns.
constexpr int kSlice = 8;

template <typename TS> struct C2Sel;
template <> struct C2Sel<double> { using type = double2; };
template <> struct C2Sel<float> { using type = float2; };
__device__ __forceinline__ void red_add(float* p, float v) { atomicAdd(p, v); }
// one complex value per reduction: a single red.global.add.v2.f32 for complex64 (8-byte aligned), two RED.ADD.F64 for complex128
__device__ __forceinline__ void red_add2(float* p, float re, float im) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(re), "f"(im) : "memory");
}
__device__ __forceinline__ void red_add2(double* p, double re, double im) { atomicAdd(p, re); atomicAdd(p + 1, im); }

// TT: arithmetic type of the contraction; TS: storage type of the multivectors (double: complex128, float: complex64)
template <typename TT, typename TS>
__global__ void __launch_bounds__(128)
proj_kernel(const NonlocalDev nl, const ProjArgs ar) {
    using S2 = typename C2Sel<TS>::type;
    const ProjItem it = nl.items[blockIdx.x];
    const int s = blockIdx.y & 1;
    const int v = (blockIdx.y >> 1) * 128 + threadIdx.x;
    if (v >= ar.nvec) return;
    const int np = nl.nproj[it.atom];
    const long long soff = nl.s_off[it.atom] + it.start;
    const long long poff = nl.p_off[it.atom] + (long long)it.start * np;
    double2 x[kSlice];
#pragma unroll
    for (int jj = 0; jj < kSlice; ++jj) {
        x[jj] = make_double2(0.0, 0.0);
        if (jj < it.count) {
            const long long I = nl.supp_node[soff + jj];
            const S2 xs = __ldg(reinterpret_cast<const S2*>(ar.in) + (2 * I + s) * ar.ld_in + v);
            x[jj] = make_double2((double)xs.x, (double)xs.y);
            { const double m = (ar.mass_u ? nl.supp_mass[soff + jj] : 1.0) * ar.in_scale; x[jj].x *= m; x[jj].y *= m; }
        }
    }
    double* Crow = ar.C + (nl.c_off[it.atom] * (long long)ar.nvec + v) * 2;
    for (int b = 0; b < np; ++b) {
        TT cr = 0, ci = 0;
#pragma unroll
        for (int jj = 0; jj < kSlice; ++jj) {
            if (jj < it.count) {
                TT pr, pi;
                if (sizeof(TT) == 8) { const double2 pv = nl.P64[poff + jj * np + b]; pr = pv.x; pi = pv.y; }
                else { const float2 pv = nl.P32[poff + jj * np + b]; pr = pv.x; pi = pv.y; }
                const TT xr = (TT)x[jj].x, xi = (TT)x[jj].y;
                cr = fma(pr, xr, fma(pi, xi, cr));                   // conj(p) x = (pr - i pi)(xr + i xi)
                ci = fma(pr, xi, fma(-pi, xr, ci));
            }
        }
        double* dst = Crow + (long long)(2 * b + s) * ar.nvec * 2;
        red_add(dst, (double)cr);
        red_add(dst + 1, (double)ci);
    }
}

// G[c_off + row][v] = sum_r D_a[row][r] C[c_off + r][v]; one thread per (row, v)
__global__ void __launch_bounds__(128)
gmat_kernel(const NonlocalDev nl, const double2* __restrict__ Cc, double2* __restrict__ G, int nvec) {
    const int atom = blockIdx.x;
    const int np2 = 2 * nl.nproj[atom];
    const int row = blockIdx.y;
    const int v = blockIdx.z * 128 + threadIdx.x;
    if (row >= np2 || v >= nvec) return;
    const double2* D = nl.D64 + nl.d_off[atom] + (long long)row * np2;
    const double2* c = Cc + nl.c_off[atom] * (long long)nvec + v;
    double gr = 0.0, gi = 0.0;
#pragma unroll 8
    for (int r = 0; r < np2; ++r) {
        const double2 d = D[r];
        const double2 cv = c[(long long)r * nvec];
        gr += d.x * cv.x - d.y * cv.y;
        gi += d.x * cv.y + d.y * cv.x;
    }
    G[(nl.c_off[atom] + row) * (long long)nvec + v] = make_double2(gr, gi);
}

template <typename TT, typename TS>
__global__ void __launch_bounds__(128)
back_kernel(const NonlocalDev nl, const BackArgs ar) {
    const ProjItem it = nl.items[blockIdx.x];
    const int s = blockIdx.y & 1;
    const int v = (blockIdx.y >> 1) * 128 + threadIdx.x;
    if (v >= ar.nvec) return;
    const int np = nl.nproj[it.atom];
    const long long soff = nl.s_off[it.atom] + it.start;
    const long long poff = nl.p_off[it.atom] + (long long)it.start * np;
    const double2* G = reinterpret_cast<const double2*>(ar.G) + nl.c_off[it.atom] * (long long)ar.nvec + v;
    TT yr[kSlice], yi[kSlice];
#pragma unroll
    for (int jj = 0; jj < kSlice; ++jj) { yr[jj] = 0; yi[jj] = 0; }
    for (int b = 0; b < np; ++b) {
        const double2 g = G[(long long)(2 * b + s) * ar.nvec];
        const TT gr = (TT)g.x, gi = (TT)g.y;
#pragma unroll
        for (int jj = 0; jj < kSlice; ++jj) {
            if (jj < it.count) {
                TT pr, pi;
                if (sizeof(TT) == 8) { const double2 pv = nl.P64[poff + jj * np + b]; pr = pv.x; pi = pv.y; }
                else { const float2 pv = nl.P32[poff + jj * np + b]; pr = pv.x; pi = pv.y; }
                yr[jj] = fma(pr, gr, fma(-pi, gi, yr[jj]));
                yi[jj] = fma(pr, gi, fma(pi, gr, yi[jj]));
            }
        }
    }
#pragma unroll
    for (int jj = 0; jj < kSlice; ++jj) {
        if (jj < it.count) {
            const long long I = nl.supp_node[soff + jj];
            const double f = ar.cH * (ar.sout_invm ? 1.0 : nl.supp_mass[soff + jj]);
            TS* dst = reinterpret_cast<TS*>(ar.out) + ((2 * I + s) * ar.ld_out + v) * 2;
            red_add(dst, (TS)(f * (double)yr[jj]));
            red_add(dst + 1, (TS)(f * (double)yi[jj]));
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Fast S4 path when every atom has the same NP projectors (NP = 4 or 8; the BASELINE configs): items of up to
// kBig = 32 support nodes, the item's projector block, node list and masses staged in shared memory once, the
// coefficients of one (spin, vector) column kept in registers across the item, so that C receives one RED per
// coefficient and item (4x fewer than the 8-node slices above) and all loads of a batch are in flight together.
// back_fast also forms its rows of G = D_a C_a itself (D_a in shared memory), which removes the gmat launch.
constexpr int kBig = 32;

template <typename TT> struct P2Sel;
template <> struct P2Sel<double> { using type = double2; static __device__ __forceinline__ const double2* ptr(const NonlocalDev& nl) { return nl.P64; } };
template <> struct P2Sel<float> { using type = float2; static __device__ __forceinline__ const float2* ptr(const NonlocalDev& nl) { return nl.P32; } };

template <typename TT, typename TS, int NP>
__global__ void __launch_bounds__(128)
proj_fast_kernel(const NonlocalDev nl, const ProjArgs ar) {
    using P2 = typename P2Sel<TT>::type;
    using S2 = typename C2Sel<TS>::type;
    __shared__ P2 Ps[kBig * NP];
    __shared__ long long nodes[kBig];
    __shared__ double mass[kBig];
    const ProjItem it = nl.items_big[blockIdx.x];
    const long long soff = nl.s_off[it.atom] + it.start;
    const long long poff = nl.p_off[it.atom] + (long long)it.start * NP;
    for (int i = threadIdx.x; i < it.count * NP; i += 128) Ps[i] = P2Sel<TT>::ptr(nl)[poff + i];
    if (threadIdx.x < kBig) {
        const int jj = threadIdx.x < it.count ? threadIdx.x : 0;
        nodes[threadIdx.x] = nl.supp_node[soff + jj];
        mass[threadIdx.x] = (ar.mass_u ? nl.supp_mass[soff + jj] : 1.0) * ar.in_scale;
    }
    __syncthreads();
    const int s = blockIdx.y & 1;
    const int v = (blockIdx.y >> 1) * 128 + threadIdx.x;
    if (v >= ar.nvec) return;
    TT cr[NP], ci[NP];
#pragma unroll
    for (int b = 0; b < NP; ++b) { cr[b] = 0; ci[b] = 0; }
    const S2* in2 = reinterpret_cast<const S2*>(ar.in) + (long long)s * ar.ld_in + v;
#pragma unroll 1
    for (int j0 = 0; j0 < it.count; j0 += kSlice) {
        S2 x[kSlice];
#pragma unroll
        for (int jj = 0; jj < kSlice; ++jj) {
            const bool ok = j0 + jj < it.count;
            x[jj].x = 0; x[jj].y = 0;
            if (ok) x[jj] = __ldg(in2 + 2 * nodes[j0 + jj] * ar.ld_in);
        }
#pragma unroll
        for (int jj = 0; jj < kSlice; ++jj) {
            if (j0 + jj < it.count) {
                const double m = mass[j0 + jj];
                const TT xr = (TT)((double)x[jj].x * m), xi = (TT)((double)x[jj].y * m);
#pragma unroll
                for (int b = 0; b < NP; ++b) {
                    const P2 pv = Ps[(j0 + jj) * NP + b];
                    cr[b] = fma(pv.x, xr, fma(pv.y, xi, cr[b]));         // conj(p) x
                    ci[b] = fma(pv.x, xi, fma(-pv.y, xr, ci[b]));
                }
            }
        }
    }
    double* Crow = ar.C + (nl.c_off[it.atom] * (long long)ar.nvec + v) * 2;
#pragma unroll
    for (int b = 0; b < NP; ++b) {
        double* dst = Crow + (long long)(2 * b + s) * ar.nvec * 2;
        red_add(dst, (double)cr[b]);
        red_add(dst + 1, (double)ci[b]);
    }
}

template <typename TT, typename TS, int NP>
__global__ void __launch_bounds__(128)
back_fast_kernel(const NonlocalDev nl, const BackArgs ar) {
    using P2 = typename P2Sel<TT>::type;
    __shared__ P2 Ps[kBig * NP];
    __shared__ double2 Ds[2 * NP * 2 * NP];
    __shared__ long long nodes[kBig];
    __shared__ double fac[kBig];
    const ProjItem it = nl.items_big[blockIdx.x];
    const long long soff = nl.s_off[it.atom] + it.start;
    const long long poff = nl.p_off[it.atom] + (long long)it.start * NP;
    for (int i = threadIdx.x; i < it.count * NP; i += 128) Ps[i] = P2Sel<TT>::ptr(nl)[poff + i];
    for (int i = threadIdx.x; i < 4 * NP * NP; i += 128) Ds[i] = nl.D64[nl.d_off[it.atom] + i];
    if (threadIdx.x < kBig) {
        const int jj = threadIdx.x < it.count ? threadIdx.x : 0;
        nodes[threadIdx.x] = nl.supp_node[soff + jj];
        fac[threadIdx.x] = ar.cH * (ar.sout_invm ? 1.0 : nl.supp_mass[soff + jj]);
    }
    __syncthreads();
    const int s = blockIdx.y & 1;
    const int v = (blockIdx.y >> 1) * 128 + threadIdx.x;
    if (v >= ar.nvec) return;
    // rows 2b + s of G = D C for this column (FP64: the coupling matrix is applied in double in every mode)
    const double2* Cc = reinterpret_cast<const double2*>(ar.C) + nl.c_off[it.atom] * (long long)ar.nvec + v;
    double gr[NP], gi[NP];
#pragma unroll
    for (int b = 0; b < NP; ++b) { gr[b] = 0.0; gi[b] = 0.0; }
#pragma unroll 4
    for (int r = 0; r < 2 * NP; ++r) {
        const double2 cv = Cc[(long long)r * ar.nvec];
#pragma unroll
        for (int b = 0; b < NP; ++b) {
            const double2 d = Ds[(2 * b + s) * 2 * NP + r];
            gr[b] = fma(d.x, cv.x, fma(-d.y, cv.y, gr[b]));
            gi[b] = fma(d.x, cv.y, fma(d.y, cv.x, gi[b]));
        }
    }
    TT g_r[NP], g_i[NP];
#pragma unroll
    for (int b = 0; b < NP; ++b) { g_r[b] = (TT)gr[b]; g_i[b] = (TT)gi[b]; }
    TS* out = reinterpret_cast<TS*>(ar.out) + ((long long)s * ar.ld_out + v) * 2;
#pragma unroll 4
    for (int jj = 0; jj < it.count; ++jj) {
        TT yr = 0, yi = 0;
#pragma unroll
        for (int b = 0; b < NP; ++b) {
            const P2 pv = Ps[jj * NP + b];
            yr = fma(pv.x, g_r[b], fma(-pv.y, g_i[b], yr));
            yi = fma(pv.x, g_i[b], fma(pv.y, g_r[b], yi));
        }
        TS* dst = out + 4 * nodes[jj] * ar.ld_out;
        red_add2(dst, (TS)(fac[jj] * (double)yr), (TS)(fac[jj] * (double)yi));
    }
}

// ---------------------------------------------------------------------------------------------
// S7 / scaled copies: out[row][v] = ca[v] * (a_inv_mass ? A/m : A) + cb[v] * B
template <typename TS>
__global__ void __launch_bounds__(256)
axpby_kernel(const __grid_constant__ MeshConst mc, double2* __restrict__ out, long long ldo,
             const typename C2Sel<TS>::type* __restrict__ A, long long lda, const double* __restrict__ ca, int a_inv_mass,
             const double2* __restrict__ B, long long ldb, const double* __restrict__ cb, int nvec) {
    const long long rows = 2 * mc.nnodes;
    const long long total = rows * nvec;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const long long row = idx / nvec;
        const int v = (int)(idx - row * nvec);
        double f = ca[v];
        if (a_inv_mass) {
            const long long I = row >> 1;
            const int ix = (int)(I % mc.n1[0]);
            const int iy = (int)((I / mc.n1[0]) % mc.n1[1]);
            const int iz = (int)(I / ((long long)mc.n1[0] * mc.n1[1]));
            f *= mc.im1[0][ix % mc.p] * mc.im1[1][iy % mc.p] * mc.im1[2][iz % mc.p];
        }
        const typename C2Sel<TS>::type av = A[row * lda + v];
        double2 r = make_double2(f * (double)av.x, f * (double)av.y);
        if (B != nullptr) {
            const double g = cb[v];
            const double2 bv = B[row * ldb + v];
            r.x = fma(g, bv.x, r.x); r.y = fma(g, bv.y, r.y);
        }
        out[row * ldo + v] = r;
    }
}

// ---------------------------------------------------------------------------------------------
// Coefficient table: one thread per vector runs the FP64 Lambda_k recurrence.
__global__ void coef_kernel(const double* __restrict__ hdr, double* __restrict__ table, int nrows, int nvec) {
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= nvec) return;
    const CoefRow* rows = reinterpret_cast<const CoefRow*>(hdr + 4);
    const double lam = hdr[4 + 9 * (size_t)nrows + v];
    double Lp = 1.0, L = hdr[0] + hdr[1] * lam;
    for (int r = 0; r < nrows; ++r) {
        const CoefRow row = rows[r];
        table[(size_t)r * 2 * nvec + v] = row.cin0 + row.cinL * L + row.cinLam * lam;
        table[(size_t)r * 2 * nvec + nvec + v] = row.cR0 + row.cRL * L;
        if (row.advance != 0.0) {
            const double Ln = row.al * lam * L - row.be * L - row.ga * Lp;
            Lp = L; L = Ln;
        }
    }
}

cudaError_t launch_coef(const double* hdr, double* table, int nrows, int nvec, cudaStream_t st) {
    coef_kernel<<<(nvec + 127) / 128, 128, 0, st>>>(hdr, table, nrows, nvec);
    count_launch();
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// launchers
template <int P, int NV, typename TT>
static cudaError_t launch_cell_t(const chfsi_mesh* m, const CellArgs& a, cudaStream_t st) {
    constexpr int n = P + 1, C = 4 * NV;
    const size_t smem = 2ull * n * n * n * C * sizeof(TT);
    static bool attr_done[64] = {false};
    auto kern = cell_kernel<P, NV, TT>;
    if (!attr_done[m->device & 63]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_done[m->device & 63] = true;
    }
    const int nchunks = (a.nvec + NV - 1) / NV;
    const long long grid = (long long)m->mc.ncells * nchunks;
    kern<<<(unsigned)grid, n * C, smem, st>>>(m->mc, a);
    return cudaGetLastError();
}

bool cell_supported(int p, chfsi_prec prec) {
    if (prec == CHFSI_FP32_STORED) return p == 2 || p == 4 || p == 6 || p == 8;   // line-owned kernel only
    if (prec == CHFSI_TF32 || prec == CHFSI_TF32X3) return p == 2 || p == 4 || p == 6 || p == 8;   // tensor-core kernel only
    if (prec != CHFSI_FP64 && prec != CHFSI_FP32) return false;
    return p >= 1 && p <= 8;
}

static cudaError_t launch_cell_legacy(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t st);

// The dominant kernel.  FP64: the z-marching kernel (cell_march.cu) for p = 2, 4, 6 (within a few percent of its memory
// floor at p = 6), the line-owned x/y/z kernel (cell_xyz.cu) for p = 8.  FP32 product and FP32-stored multivectors: the
// line-owned kernel.  Odd degrees: the tile-per-cell kernel above.
cudaError_t launch_cell(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t st) {
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (m->prof_on) {
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return cudaGetLastError();
        cudaEventRecord(e0, st);
    }
    cudaError_t err;
    const int choice = m->cell_kernel[(int)prec];             // chfsi_mesh_set_cell_kernel; 0 = the library's choice
    const bool tf = prec == CHFSI_TF32 || prec == CHFSI_TF32X3;
    const bool use_mma = (tf || (prec == CHFSI_FP64 && choice == CHFSI_CELL_MMA)) && mma_supported(m, prec, a);
    const bool use_march = !use_mma && prec == CHFSI_FP64 && (choice == CHFSI_CELL_MARCH || (choice == 0 && m->p <= 6)) &&
                           march_supported(m, prec, a);
    if (use_mma) err = launch_cell_mma(m, prec, a, st);
    else if (tf) err = cudaErrorInvalidValue;
    else if (!use_march && xyz_supported(m, prec, a)) err = launch_cell_xyz(m, prec, a, st);
    else if (use_march) err = launch_cell_march(m, prec, a, st);
    else if (a.store_f32) err = cudaErrorInvalidValue;
    else err = launch_cell_legacy(m, prec, a, st);
    count_launch();
    if (m->prof_on) {
        cudaEventRecord(e1, st);
        m->prof_ev.push_back(e0); m->prof_ev.push_back(e1);
        // algorithmic bytes per unit: `in` read once, `out` read and written by the reduction, R read in FP64
        const double eb = a.store_f32 ? 8.0 : 16.0;
        m->prof_bytes += 2.0 * (double)m->nnodes * a.nvec * (eb + 2.0 * eb + ((a.R != nullptr && a.cR != nullptr) ? 16.0 : 0.0));
    }
    return err;
}

static cudaError_t launch_cell_legacy(const chfsi_mesh* m, chfsi_prec prec, const CellArgs& a, cudaStream_t st) {
    const bool f32 = prec == CHFSI_FP32;
#define CELL_CASE(PP, NV64, NV32)                                                     \
    case PP:                                                                           \
        return f32 ? launch_cell_t<PP, NV32, float>(m, a, st) : launch_cell_t<PP, NV64, double>(m, a, st);
    switch (m->p) {
        CELL_CASE(1, 8, 8)
        CELL_CASE(2, 8, 8)
        CELL_CASE(3, 8, 8)
        CELL_CASE(4, 8, 8)
        CELL_CASE(5, 8, 8)
        CELL_CASE(6, 4, 8)
        CELL_CASE(7, 4, 8)
        CELL_CASE(8, 4, 4)
        default: return cudaErrorInvalidValue;
    }
#undef CELL_CASE
}

template <typename TT, typename TS>
static void launch_proj_t(const chfsi_mesh* m, const ProjArgs& a, cudaStream_t st) {
    if (m->nl.uniform_np == 4 || m->nl.uniform_np == 8) {
        dim3 grid(m->nl.nitems_big, 2 * ((a.nvec + 127) / 128));
        if (m->nl.uniform_np == 8) proj_fast_kernel<TT, TS, 8><<<grid, 128, 0, st>>>(m->nl, a);
        else proj_fast_kernel<TT, TS, 4><<<grid, 128, 0, st>>>(m->nl, a);
    } else {
        dim3 grid(m->nl.nitems, 2 * ((a.nvec + 127) / 128));
        proj_kernel<TT, TS><<<grid, 128, 0, st>>>(m->nl, a);
    }
}

cudaError_t launch_proj(const chfsi_mesh* m, chfsi_prec prec, const ProjArgs& a, cudaStream_t st) {
    if (m->nl.nitems == 0) return cudaSuccess;
    if (a.store_f32) launch_proj_t<float, float>(m, a, st);
    else if (prec == CHFSI_FP64) launch_proj_t<double, double>(m, a, st);
    else launch_proj_t<float, double>(m, a, st);
    count_launch();
    return cudaGetLastError();
}

template <typename TT, typename TS>
static void launch_back_t(const chfsi_mesh* m, const BackArgs& a, cudaStream_t st) {
    if (m->nl.uniform_np == 4 || m->nl.uniform_np == 8) {
        dim3 grid(m->nl.nitems_big, 2 * ((a.nvec + 127) / 128));
        if (m->nl.uniform_np == 8) back_fast_kernel<TT, TS, 8><<<grid, 128, 0, st>>>(m->nl, a);
        else back_fast_kernel<TT, TS, 4><<<grid, 128, 0, st>>>(m->nl, a);
        return;
    }
    {
        dim3 gg(m->nl.natoms, 2 * m->nl.max_nproj, (a.nvec + 127) / 128);
        gmat_kernel<<<gg, 128, 0, st>>>(m->nl, reinterpret_cast<const double2*>(a.C), reinterpret_cast<double2*>(a.G), a.nvec);
        count_launch();
    }
    dim3 grid(m->nl.nitems, 2 * ((a.nvec + 127) / 128));
    back_kernel<TT, TS><<<grid, 128, 0, st>>>(m->nl, a);
}

cudaError_t launch_back(const chfsi_mesh* m, chfsi_prec prec, const BackArgs& a, cudaStream_t st) {
    if (m->nl.nitems == 0) return cudaSuccess;
    if (a.store_f32) launch_back_t<float, float>(m, a, st);
    else if (prec == CHFSI_FP64) launch_back_t<double, double>(m, a, st);
    else launch_back_t<float, double>(m, a, st);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_axpby(const chfsi_mesh* m, double* out, long long ldo, const void* A, long long lda, int a_f32,
                         const double* ca, int a_inv_mass, const double* B, long long ldb,
                         const double* cb, int nvec, cudaStream_t st) {
    const long long total = 2 * m->nnodes * (long long)nvec;
    long long blocks = (total + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (a_f32)
        axpby_kernel<float><<<(unsigned)blocks, 256, 0, st>>>(m->mc, reinterpret_cast<double2*>(out), ldo,
                                                              reinterpret_cast<const float2*>(A), lda, ca, a_inv_mass,
                                                              reinterpret_cast<const double2*>(B), ldb, cb, nvec);
    else
        axpby_kernel<double><<<(unsigned)blocks, 256, 0, st>>>(m->mc, reinterpret_cast<double2*>(out), ldo,
                                                               reinterpret_cast<const double2*>(A), lda, ca, a_inv_mass,
                                                               reinterpret_cast<const double2*>(B), ldb, cb, nvec);
    count_launch();
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// FP32-stored multivectors (CHFSI_FP32_STORED): the FP32 copy of Zh_1 = R, and the power-of-two renormalisation of the
// scaled iterates (both streaming, a few times per filter call)
__global__ void __launch_bounds__(256)
cast32_kernel(float2* __restrict__ dst, long long ldd, const double2* __restrict__ src, long long lds, long long rows, int nvec) {
    const long long total = rows * nvec;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const long long row = idx / nvec;
        const int v = (int)(idx - row * nvec);
        const double2 s = src[row * lds + v];
        dst[row * ldd + v] = make_float2((float)s.x, (float)s.y);
    }
}

template <typename T>
__global__ void __launch_bounds__(256)
scale_kernel(T* __restrict__ buf, long long count, T f) {
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < count; idx += (long long)gridDim.x * blockDim.x)
        buf[idx] *= f;
}

cudaError_t launch_cast32(const chfsi_mesh* m, void* dst, long long ldd, const double* src, long long lds, int nvec, cudaStream_t st) {
    const long long total = 2 * m->nnodes * (long long)nvec;
    long long blocks = (total + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    cast32_kernel<<<(unsigned)blocks, 256, 0, st>>>(reinterpret_cast<float2*>(dst), ldd, reinterpret_cast<const double2*>(src), lds,
                                                    2 * m->nnodes, nvec);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_scale(const chfsi_mesh* m, void* buf, int f32, int nvec, double f, cudaStream_t st) {
    const long long count = 4 * m->nnodes * (long long)nvec;     // reals
    long long blocks = (count + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (f32) scale_kernel<float><<<(unsigned)blocks, 256, 0, st>>>(reinterpret_cast<float*>(buf), count, (float)f);
    else scale_kernel<double><<<(unsigned)blocks, 256, 0, st>>>(reinterpret_cast<double*>(buf), count, f);
    count_launch();
    return cudaGetLastError();
}

}  // namespace chfsi
