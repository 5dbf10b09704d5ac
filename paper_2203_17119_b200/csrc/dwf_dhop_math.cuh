// Per-leg arithmetic of the Wilson hopping term, shared by the Dhop kernels (readings C1, C3, C10):
// 128-bit vector types, link load + third-row reconstruction, spin projection, SU(3) x half-spinor,
// reconstruct-accumulate.  Chiral basis, gamma5 = diag(1,1,-1,-1).
#pragma once
#include "dwf_layout.cuh"

namespace dwf {

template <typename R> struct VT;
template <> struct VT<float> { using V = float4; static constexpr int VW = 4, K = 6; };
template <> struct VT<double> { using V = double2; static constexpr int VW = 2, K = 12; };

__device__ __forceinline__ void unpackv(const float4& v, float* d) { d[0] = v.x; d[1] = v.y; d[2] = v.z; d[3] = v.w; }
__device__ __forceinline__ void unpackv(const double2& v, double* d) { d[0] = v.x; d[1] = v.y; }
__device__ __forceinline__ float4 packv(const float* d) { return make_float4(d[0], d[1], d[2], d[3]); }
__device__ __forceinline__ double2 packv(const double* d) { return make_double2(d[0], d[1]); }

__device__ __forceinline__ float4 ldg_v(const float4* p) { return __ldg(p); }
__device__ __forceinline__ double2 ldg_v(const double2* p) { return __ldg(p); }

// ---- link load: NG = 12 (rows 0,1; row 2 = conj(row0 x row1), reading C10) or 18 --------------
// native gauge: 16-byte vectors, vec index = ((tile*8 + leg)*KG + kg)*TS + lane
template <typename R, int NG>
__device__ __forceinline__ void load_link(const typename VT<R>::V* __restrict__ Wp, int TS, R (&u)[18]) {
    constexpr int VW = VT<R>::VW;
    constexpr int KG = (NG + VW - 1) / VW;      // fp32/18 reals: 5 vectors, last one half used
    R tmp[KG * VW];
#pragma unroll
    for (int k = 0; k < KG; ++k) unpackv(ldg_v(Wp + (size_t)k * TS), tmp + k * VW);
#pragma unroll
    for (int i = 0; i < NG; ++i) u[i] = tmp[i];
    if (NG == 12) {
        // row2[c] = conj( row0[a]*row1[b] - row0[b]*row1[a] ), (a,b) cyclic after c
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int a = (c + 1) % 3, b = (c + 2) % 3;
            R ar = u[2 * a], ai = u[2 * a + 1], br = u[6 + 2 * b], bi = u[6 + 2 * b + 1];
            R cr = u[2 * b], ci = u[2 * b + 1], dr = u[6 + 2 * a], di = u[6 + 2 * a + 1];
            R re = (ar * br - ai * bi) - (cr * dr - ci * di);
            R im = (ar * bi + ai * br) - (cr * di + ci * dr);
            u[12 + 2 * c] = re;
            u[12 + 2 * c + 1] = -im;
        }
    }
}

// row 2 of an SU(3) link from rows 0, 1 (reading C10): u[12..17] = conj(row0 x row1)
template <typename R>
__device__ __forceinline__ void third_row(R (&u)[18]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        R ar = u[2 * a], ai = u[2 * a + 1], br = u[6 + 2 * b], bi = u[6 + 2 * b + 1];
        R cr = u[2 * b], ci = u[2 * b + 1], dr = u[6 + 2 * a], di = u[6 + 2 * a + 1];
        u[12 + 2 * c] = (ar * br - ai * bi) - (cr * dr - ci * di);
        u[12 + 2 * c + 1] = -((ar * bi + ai * br) - (cr * di + ci * dr));
    }
}

// ---- spin projection: h = upper two rows of (1 + SG*gamma_MU) psi ------------------------------
// psi[(sp*3+c)*2+ri]; h[(hs*3+c)*2+ri]
template <typename R, int MU, int SG>
__device__ __forceinline__ void spin_project(const R (&psi)[24], R (&h)[12]) {
    constexpr R s = (R)SG;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int p0 = 2 * c, p1 = 6 + 2 * c, p2 = 12 + 2 * c, p3 = 18 + 2 * c;
        const int h0 = 2 * c, h1 = 6 + 2 * c;
        if (MU == 0) {          // h0 = psi0 + s*i*psi3 ; h1 = psi1 + s*i*psi2
            h[h0] = psi[p0] - s * psi[p3 + 1]; h[h0 + 1] = psi[p0 + 1] + s * psi[p3];
            h[h1] = psi[p1] - s * psi[p2 + 1]; h[h1 + 1] = psi[p1 + 1] + s * psi[p2];
        } else if (MU == 1) {   // h0 = psi0 - s*psi3 ; h1 = psi1 + s*psi2
            h[h0] = psi[p0] - s * psi[p3]; h[h0 + 1] = psi[p0 + 1] - s * psi[p3 + 1];
            h[h1] = psi[p1] + s * psi[p2]; h[h1 + 1] = psi[p1 + 1] + s * psi[p2 + 1];
        } else if (MU == 2) {   // h0 = psi0 + s*i*psi2 ; h1 = psi1 - s*i*psi3
            h[h0] = psi[p0] - s * psi[p2 + 1]; h[h0 + 1] = psi[p0 + 1] + s * psi[p2];
            h[h1] = psi[p1] + s * psi[p3 + 1]; h[h1 + 1] = psi[p1 + 1] - s * psi[p3];
        } else {                // h0 = psi0 + s*psi2 ; h1 = psi1 + s*psi3
            h[h0] = psi[p0] + s * psi[p2]; h[h0 + 1] = psi[p0 + 1] + s * psi[p2 + 1];
            h[h1] = psi[p1] + s * psi[p3]; h[h1 + 1] = psi[p1 + 1] + s * psi[p3 + 1];
        }
    }
}

// ---- g = W h (3x3 complex times two colour vectors) -------------------------------------------
template <typename R>
__device__ __forceinline__ void su3_mul(const R (&u)[18], const R (&h)[12], R (&g)[12]) {
#pragma unroll
    for (int hs = 0; hs < 2; ++hs)
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            R re = u[(r * 3) * 2] * h[hs * 6] - u[(r * 3) * 2 + 1] * h[hs * 6 + 1];
            R im = u[(r * 3) * 2] * h[hs * 6 + 1] + u[(r * 3) * 2 + 1] * h[hs * 6];
#pragma unroll
            for (int c = 1; c < 3; ++c) {
                const R wr = u[(r * 3 + c) * 2], wi = u[(r * 3 + c) * 2 + 1];
                const R hr = h[hs * 6 + 2 * c], hi = h[hs * 6 + 2 * c + 1];
                re += wr * hr; re -= wi * hi;
                im += wr * hi; im += wi * hr;
            }
            g[hs * 6 + 2 * r] = re;
            g[hs * 6 + 2 * r + 1] = im;
        }
}

// ---- acc += reconstruct((1 + SG*gamma_MU) from g) ---------------------------------------------
template <typename R, int MU, int SG>
__device__ __forceinline__ void spin_recon_acc(const R (&g)[12], R (&acc)[24]) {
    constexpr R s = (R)SG;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int g0 = 2 * c, g1 = 6 + 2 * c;
        const int a0 = 2 * c, a1 = 6 + 2 * c, a2 = 12 + 2 * c, a3 = 18 + 2 * c;
        acc[a0] += g[g0]; acc[a0 + 1] += g[g0 + 1];
        acc[a1] += g[g1]; acc[a1 + 1] += g[g1 + 1];
        if (MU == 0) {          // row2 = -s*i*g1 ; row3 = -s*i*g0
            acc[a2] += s * g[g1 + 1]; acc[a2 + 1] -= s * g[g1];
            acc[a3] += s * g[g0 + 1]; acc[a3 + 1] -= s * g[g0];
        } else if (MU == 1) {   // row2 = s*g1 ; row3 = -s*g0
            acc[a2] += s * g[g1]; acc[a2 + 1] += s * g[g1 + 1];
            acc[a3] -= s * g[g0]; acc[a3 + 1] -= s * g[g0 + 1];
        } else if (MU == 2) {   // row2 = -s*i*g0 ; row3 = s*i*g1
            acc[a2] += s * g[g0 + 1]; acc[a2 + 1] -= s * g[g0];
            acc[a3] -= s * g[g1 + 1]; acc[a3 + 1] += s * g[g1];
        } else {                // row2 = s*g0 ; row3 = s*g1
            acc[a2] += s * g[g0]; acc[a2 + 1] += s * g[g0 + 1];
            acc[a3] += s * g[g1]; acc[a3 + 1] += s * g[g1 + 1];
        }
    }
}

}  // namespace dwf
