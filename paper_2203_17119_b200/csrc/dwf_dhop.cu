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
#include "dwf_dhop_math.cuh"

namespace dwf {

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
    const Geom g = geom_prec(c, sizeof(R) == 8 ? DWF_F64 : DWF_F32, c->nrhs_cur);
    const int nchunks = (g.Ls + SC - 1) / SC;
    int block = 128;
    if (g.TS < block) block = ((g.TS + 31) / 32) * 32;
    dim3 grid((g.Vh + block - 1) / block, nchunks);
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
        default: c->err = "dhop: slices per thread must be 1..4"; return DWF_EINVAL;
    }
}

dwf_status dhop_timing_flush(dwf_ctx* c) {
    if (c->ev_used == 0) return DWF_OK;
    DWF_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    for (int i = 0; i < c->ev_used; i += 2) {
        float ms = 0.f;
        DWF_CUDA_CHECK(c, cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]));
        c->dhop_ms += ms;
        c->dhop_timed++;
    }
    c->ev_used = 0;
    return DWF_OK;
}

static dwf_status launch_dhop_untimed(dwf_ctx* c, void* out, const void* in, int out_parity, int dagger, int prec);

// per-launch CUDA-event timing of the Dhop kernels ("time_dhop"): events on the launching stream around the launch;
// alg_bytes = algorithmic bytes of this launch, summed for bench.py's roofline
dwf_status dhop_time_begin(dwf_ctx* c) {
    if (!c->time_dhop) return DWF_OK;
    const int POOL = 2048;
    if (c->ev.empty()) {
        c->ev.resize(POOL);
        for (int i = 0; i < POOL; ++i) DWF_CUDA_CHECK(c, cudaEventCreate(&c->ev[i]));
    }
    if (c->ev_used + 2 > POOL) {
        dwf_status st = dhop_timing_flush(c);
        if (st != DWF_OK) return st;
    }
    DWF_CUDA_CHECK(c, cudaEventRecord(c->ev[c->ev_used], c->stream));
    return DWF_OK;
}
dwf_status dhop_time_end(dwf_ctx* c, double alg_bytes) {
    if (!c->time_dhop) return DWF_OK;
    DWF_CUDA_CHECK(c, cudaEventRecord(c->ev[c->ev_used + 1], c->stream));
    c->ev_used += 2;
    c->dhop_bytes += alg_bytes;
    return DWF_OK;
}

// half-field Dhop: out has parity out_parity, in has the other parity
dwf_status launch_dhop(dwf_ctx* c, void* out, const void* in, int out_parity, int dagger, int prec) {
    dwf_status st = dhop_time_begin(c);
    if (st != DWF_OK) return st;
    st = launch_dhop_untimed(c, out, in, out_parity, dagger, prec);
    if (st != DWF_OK) return st;
    const double B = (prec == DWF_F64) ? 8.0 : 4.0;
    // algorithmic bytes: every system's field in and out, the links once for all of them
    return dhop_time_end(c, 2.0 * half_bytes(c->g, prec) * c->nrhs_cur + (double)c->g.Vh * 8 * (c->compress12 ? 12 : 18) * B);
}

static dwf_status launch_dhop_untimed(dwf_ctx* c, void* out, const void* in, int out_parity, int dagger, int prec) {
    if (c->dhop_kernel == 0) {
        bool handled = false;
        dwf_status st = launch_dhop_tma(c, out, in, out_parity, dagger, prec, &handled);
        if (st != DWF_OK || handled) return st;
    }
    if (c->dhop_kernel != 1) {
        bool handled = false;
        dwf_status st = launch_dhop_pipe(c, out, in, out_parity, dagger, prec, &handled);
        if (st != DWF_OK || handled) return st;
    }
    const void* W = (prec == DWF_F64) ? c->W64[out_parity] : c->W32[out_parity];
    const int sc = (prec == DWF_F64) ? 2 : 4;       // s slices per thread
    if (prec == DWF_F64)
        return c->compress12 ? launch_sc<double, 12>(c, out, in, W, out_parity, dagger, sc)
                             : launch_sc<double, 18>(c, out, in, W, out_parity, dagger, sc);
    return c->compress12 ? launch_sc<float, 12>(c, out, in, W, out_parity, dagger, sc)
                         : launch_sc<float, 18>(c, out, in, W, out_parity, dagger, sc);
}

}  // namespace dwf
