// Dhop: the 4-D Wilson hopping stencil applied to all Ls slices (reading C3).
//
//   out(x,s) = sum_mu [ (1 - g_mu) U_mu(x) in(x+mu,s) + (1 + g_mu) U_mu(x-mu)^dag in(x-mu,s) ]
//
// One thread owns one 4-D output site.  For each of the 8 legs it loads the leg's link once
// (2-row compressed, third row rebuilt in registers), then streams SC fifth-dimension slices of
// the neighbour's spinor through spin-project -> SU(3) multiply -> reconstruct-accumulate, so a
// link load and its reconstruction are amortised over SC slices.  The tiled site order keeps the
// 8-fold neighbour reuse inside one CTA's L1 footprint; loads are 128-bit and coalesced over the
// lanes of a tile.  Half-spinor tables: chiral basis, gamma5 = diag(1,1,-1,-1) (reading C1).
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

template <typename R, int SC, int NG, int LEG, bool DAG>
__device__ __forceinline__ void dhop_leg(const typename VT<R>::V* __restrict__ in_nb,
                                         const typename VT<R>::V* __restrict__ Wleg, R bsign, int ns, int TS,
                                         R (&acc)[SC][24]) {
    using V = typename VT<R>::V;
    constexpr int K = VT<R>::K, VW = VT<R>::VW;
    constexpr int MU = LEG >> 1, DIR = LEG & 1;
    // forward leg carries (1 - gamma), backward (1 + gamma); dagger swaps them
    constexpr int SG = ((DIR == 0) ? -1 : +1) * (DAG ? -1 : +1);
    R u[18];
    load_link<R, NG>(Wleg, TS, u);
    if (MU == 3) {
#pragma unroll
        for (int i = 0; i < 18; ++i) u[i] *= bsign;
    }
#pragma unroll
    for (int j = 0; j < SC; ++j) {
        if (j < ns) {
            R psi[24];
            const V* p = in_nb + (size_t)j * K * TS;
#pragma unroll
            for (int k = 0; k < K; ++k) unpackv(ldg_v(p + (size_t)k * TS), psi + k * VW);
            R h[12], gg[12];
            spin_project<R, MU, SG>(psi, h);
            su3_mul<R>(u, h, gg);
            spin_recon_acc<R, MU, SG>(gg, acc[j]);
        }
    }
}

template <typename R, int SC, int NG, bool DAG>
__global__ void __launch_bounds__(256) dhop_kernel(Geom g, const typename VT<R>::V* __restrict__ in,
                                                   typename VT<R>::V* __restrict__ out,
                                                   const typename VT<R>::V* __restrict__ W, int out_parity,
                                                   int nchunks) {
    using V = typename VT<R>::V;
    constexpr int K = VT<R>::K, VW = VT<R>::VW;
    constexpr int KG = (NG + VW - 1) / VW;
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= g.Vh) return;
    const int TS = g.TS, Ls = g.Ls;
    const int tile = gid / TS, lane = gid - tile * TS;
    const Coord c = site_coords(g, tile, lane, out_parity);

    // neighbour base offsets (vec units, s = 0, k = 0) for the 8 legs
    unsigned nb[8];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        int y[4] = {c.x[0], c.x[1], c.x[2], c.x[3]};
        int t2, l2;
        y[mu] = c.x[mu] + 1; if (y[mu] == g.L[mu]) y[mu] = 0;
        native_site(g, y, t2, l2);
        nb[2 * mu] = (unsigned)t2 * (unsigned)(Ls * K * TS) + (unsigned)l2;
        y[mu] = c.x[mu] - 1; if (y[mu] < 0) y[mu] = g.L[mu] - 1;
        native_site(g, y, t2, l2);
        nb[2 * mu + 1] = (unsigned)t2 * (unsigned)(Ls * K * TS) + (unsigned)l2;
    }
    const R bs_f = (g.antiperiodic_t && c.x[3] == g.L[3] - 1) ? (R)-1 : (R)1;
    const R bs_b = (g.antiperiodic_t && c.x[3] == 0) ? (R)-1 : (R)1;
    const V* Wt = W + (size_t)tile * 8 * KG * TS + lane;
    V* outp = out + (size_t)tile * Ls * K * TS + lane;
    const size_t strideS = (size_t)K * TS;

    for (int chunk = blockIdx.y; chunk < nchunks; chunk += gridDim.y) {
        const int s0 = chunk * SC;
        const int ns = min(SC, Ls - s0);
        R acc[SC][24];
#pragma unroll
        for (int j = 0; j < SC; ++j)
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[j][i] = (R)0;
        const size_t so = (size_t)s0 * strideS;
        dhop_leg<R, SC, NG, 0, DAG>(in + nb[0] + so, Wt + (size_t)0 * KG * TS, (R)1, ns, TS, acc);
        dhop_leg<R, SC, NG, 1, DAG>(in + nb[1] + so, Wt + (size_t)1 * KG * TS, (R)1, ns, TS, acc);
        dhop_leg<R, SC, NG, 2, DAG>(in + nb[2] + so, Wt + (size_t)2 * KG * TS, (R)1, ns, TS, acc);
        dhop_leg<R, SC, NG, 3, DAG>(in + nb[3] + so, Wt + (size_t)3 * KG * TS, (R)1, ns, TS, acc);
        dhop_leg<R, SC, NG, 4, DAG>(in + nb[4] + so, Wt + (size_t)4 * KG * TS, (R)1, ns, TS, acc);
        dhop_leg<R, SC, NG, 5, DAG>(in + nb[5] + so, Wt + (size_t)5 * KG * TS, (R)1, ns, TS, acc);
        dhop_leg<R, SC, NG, 6, DAG>(in + nb[6] + so, Wt + (size_t)6 * KG * TS, bs_f, ns, TS, acc);
        dhop_leg<R, SC, NG, 7, DAG>(in + nb[7] + so, Wt + (size_t)7 * KG * TS, bs_b, ns, TS, acc);
#pragma unroll
        for (int j = 0; j < SC; ++j) {
            if (j < ns) {
                V* o = outp + so + (size_t)j * strideS;
#pragma unroll
                for (int k = 0; k < K; ++k) o[(size_t)k * TS] = packv(acc[j] + k * VW);
            }
        }
    }
}

template <typename R, int SC, int NG>
static dwf_status launch_t(dwf_ctx* c, void* out, const void* in, const void* W, int out_parity, int dagger) {
    using V = typename VT<R>::V;
    const Geom& g = c->g;
    const int nchunks = (g.Ls + SC - 1) / SC;
    int block = 128;
    if (g.TS < block) block = ((g.TS + 31) / 32) * 32;
    dim3 grid((g.Vh + block - 1) / block, c->dhop_loop_s ? 1 : nchunks);
    if (dagger)
        dhop_kernel<R, SC, NG, true><<<grid, block, 0, c->stream>>>(g, (const V*)in, (V*)out, (const V*)W, out_parity, nchunks);
    else
        dhop_kernel<R, SC, NG, false><<<grid, block, 0, c->stream>>>(g, (const V*)in, (V*)out, (const V*)W, out_parity, nchunks);
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

template <typename R, int NG>
static dwf_status launch_sc(dwf_ctx* c, void* out, const void* in, const void* W, int out_parity, int dagger, int sc) {
    switch (sc) {
        case 1: return launch_t<R, 1, NG>(c, out, in, W, out_parity, dagger);
        case 2: return launch_t<R, 2, NG>(c, out, in, W, out_parity, dagger);
        case 3: return launch_t<R, 3, NG>(c, out, in, W, out_parity, dagger);
        case 4: return launch_t<R, 4, NG>(c, out, in, W, out_parity, dagger);
        default: c->err = "dhop_sc must be 1..4"; return DWF_EINVAL;
    }
}

// half-field Dhop: out has parity out_parity, in has the other parity
dwf_status launch_dhop(dwf_ctx* c, void* out, const void* in, int out_parity, int dagger, int prec) {
    const void* W = (prec == DWF_F64) ? c->W64[out_parity] : c->W32[out_parity];
    int sc = c->dhop_sc;
    if (sc <= 0) sc = (prec == DWF_F64) ? 2 : 4;
    if (prec == DWF_F64)
        return c->compress12 ? launch_sc<double, 12>(c, out, in, W, out_parity, dagger, sc)
                             : launch_sc<double, 18>(c, out, in, W, out_parity, dagger, sc);
    return c->compress12 ? launch_sc<float, 12>(c, out, in, W, out_parity, dagger, sc)
                         : launch_sc<float, 18>(c, out, in, W, out_parity, dagger, sc);
}

}  // namespace dwf
