// Dhop, cp.async-pipelined tile kernel: the fallback for tile shapes and link formats the TMA kernel (dwf_dhop_tma.cu, the
// fast path on 4^4 tiles with 2-row links) does not take; dwf_dhop.cu keeps the shape-generic kernel.
//
// One CTA owns one native tile (TS output sites of one parity) for ALL Ls slices:
//   * every thread keeps its links in REGISTERS for the whole s loop (third row rebuilt once, the
//     antiperiodic sign folded in once), so a link is fetched once per 4-D site and reused Ls times
//     (north_star: "Ls innermost so each gauge link is reused Ls times");
//   * the s-slice working set of the tile -- its TS interior input sites plus the 8 halo faces of the
//     neighbouring tiles, NSLOT sites in all -- is staged in shared memory by cp.async (16-byte, L1
//     bypassed) through an NST-deep ring, two slices ahead of the arithmetic, so HBM/L2 latency is hidden
//     by the copies in flight and not by occupancy; each input site crosses L2->SM once per tile instead
//     of once per leg;
//   * threads read neighbour spinors from the stage with conflict-free 128-bit LDS ([k][slot] layout),
//     spin-project, multiply, reconstruct-accumulate, and store 128-bit coalesced.
// TPS = 1: one thread per site, 8 links in registers (fp32).  TPS = 2: two lanes (l, l^16) per site, the
// forward legs on one, the backward legs on the other (same instruction stream: the projector sign is data),
// partial sums exchanged with warp shuffles (fp64: 4 links of 18 doubles per thread).
#include <algorithm>
#include <cstdint>
#include <vector>

#include "dwf_dhop_math.cuh"

namespace dwf {

// ------------------------------------------------------------------------------------------ host tables
// For output parity p: nbslot[p][leg][lane] = stage slot holding the leg's neighbour of output site `lane`;
// slot < TS: interior (input site of the same tile, slot = its lane); slot >= TS: halo, copied from lane
// slot_lane[p][slot] of the neighbouring tile in direction slot_dir[p][slot] (leg numbering 2*mu+dir).
struct PipeTables {
    int nslot = 0;
    std::vector<uint16_t> nbslot;     // [2][8][TS]
    std::vector<int16_t> slot_dir;    // [2][nslot]  (-1 = interior)
    std::vector<uint16_t> slot_lane;  // [2][nslot]
};

static int lane_of_local(const Geom& g, const int y[4]) { return lane_from_local(g, y); }

static PipeTables build_pipe_tables(const Geom& g) {
    PipeTables t;
    const int TS = g.TS;
    int face[8], off[8], nh = 0;
    for (int d = 0; d < 8; ++d) { face[d] = TS / g.T[d >> 1]; off[d] = nh; nh += face[d]; }
    t.nslot = TS + nh;
    t.nbslot.assign((size_t)2 * 8 * TS, 0);
    t.slot_dir.assign((size_t)2 * t.nslot, -1);
    t.slot_lane.assign((size_t)2 * t.nslot, 0);
    for (int p = 0; p < 2; ++p) {
        std::vector<std::vector<int>> src(8);   // source lanes per face
        std::vector<int> want((size_t)8 * TS, -1);
        for (int lane = 0; lane < TS; ++lane) {
            int x[4];
            local_from_lane(g, lane, p, x);
            t.slot_lane[(size_t)p * t.nslot + lane] = (uint16_t)lane;
            for (int leg = 0; leg < 8; ++leg) {
                const int mu = leg >> 1;
                int y[4] = {x[0], x[1], x[2], x[3]};
                y[mu] += (leg & 1) ? -1 : +1;
                if (y[mu] >= 0 && y[mu] < g.T[mu]) {
                    t.nbslot[((size_t)p * 8 + leg) * TS + lane] = (uint16_t)lane_of_local(g, y);
                } else {
                    y[mu] = (y[mu] + g.T[mu]) % g.T[mu];
                    const int sl = lane_of_local(g, y);
                    want[(size_t)leg * TS + lane] = sl;
                    src[leg].push_back(sl);
                }
            }
        }
        for (int d = 0; d < 8; ++d) {
            std::sort(src[d].begin(), src[d].end());
            for (size_t i = 0; i < src[d].size(); ++i) {
                const int slot = TS + off[d] + (int)i;
                t.slot_dir[(size_t)p * t.nslot + slot] = (int16_t)d;
                t.slot_lane[(size_t)p * t.nslot + slot] = (uint16_t)src[d][i];
            }
            for (int lane = 0; lane < TS; ++lane) {
                const int sl = want[(size_t)d * TS + lane];
                if (sl < 0) continue;
                const int rank = (int)(std::lower_bound(src[d].begin(), src[d].end(), sl) - src[d].begin());
                t.nbslot[((size_t)p * 8 + d) * TS + lane] = (uint16_t)(TS + off[d] + rank);
            }
        }
    }
    return t;
}

// device copies live in the context (dwf_internal.h: pipe_*)
dwf_status pipe_tables_upload(dwf_ctx* c) {
    pipe_tables_free(c);
    for (int mu = 0; mu < 4; ++mu)
        if (c->g.T[mu] & 1) return DWF_OK;       // odd tile extents: generic kernel only
    for (int pr = 0; pr < 2; ++pr) {            // 0: fp32 fields, 1: fp64 fields (lane orders differ, geom_prec)
        PipeTables t = build_pipe_tables(geom_prec(c, pr ? DWF_F64 : DWF_F32));
        c->pipe_nslot = t.nslot;
        DWF_CUDA_CHECK(c, cudaMalloc(&c->pipe_nbslot[pr], t.nbslot.size() * sizeof(uint16_t)));
        DWF_CUDA_CHECK(c, cudaMalloc(&c->pipe_slot_dir[pr], t.slot_dir.size() * sizeof(int16_t)));
        DWF_CUDA_CHECK(c, cudaMalloc(&c->pipe_slot_lane[pr], t.slot_lane.size() * sizeof(uint16_t)));
        DWF_CUDA_CHECK(c, cudaMemcpy(c->pipe_nbslot[pr], t.nbslot.data(), t.nbslot.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
        DWF_CUDA_CHECK(c, cudaMemcpy(c->pipe_slot_dir[pr], t.slot_dir.data(), t.slot_dir.size() * sizeof(int16_t), cudaMemcpyHostToDevice));
        DWF_CUDA_CHECK(c, cudaMemcpy(c->pipe_slot_lane[pr], t.slot_lane.data(), t.slot_lane.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
    }
    return DWF_OK;
}

void pipe_tables_free(dwf_ctx* c) {
    for (int pr = 0; pr < 2; ++pr) {
        if (c->pipe_nbslot[pr]) cudaFree(c->pipe_nbslot[pr]);
        if (c->pipe_slot_dir[pr]) cudaFree(c->pipe_slot_dir[pr]);
        if (c->pipe_slot_lane[pr]) cudaFree(c->pipe_slot_lane[pr]);
        c->pipe_nbslot[pr] = nullptr; c->pipe_slot_dir[pr] = nullptr; c->pipe_slot_lane[pr] = nullptr;
    }
    c->pipe_nslot = 0;
}

// ------------------------------------------------------------------------------------------ device
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// h = upper two rows of (1 + s*gamma_MU) psi, s = +-1 at run time (FMA form)
template <typename R, int MU>
__device__ __forceinline__ void spin_project_s(const R (&psi)[24], R s, R (&h)[12]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int p0 = 2 * c, p1 = 6 + 2 * c, p2 = 12 + 2 * c, p3 = 18 + 2 * c;
        const int h0 = 2 * c, h1 = 6 + 2 * c;
        if (MU == 0) {
            h[h0] = psi[p0] - s * psi[p3 + 1]; h[h0 + 1] = psi[p0 + 1] + s * psi[p3];
            h[h1] = psi[p1] - s * psi[p2 + 1]; h[h1 + 1] = psi[p1 + 1] + s * psi[p2];
        } else if (MU == 1) {
            h[h0] = psi[p0] - s * psi[p3]; h[h0 + 1] = psi[p0 + 1] - s * psi[p3 + 1];
            h[h1] = psi[p1] + s * psi[p2]; h[h1 + 1] = psi[p1 + 1] + s * psi[p2 + 1];
        } else if (MU == 2) {
            h[h0] = psi[p0] - s * psi[p2 + 1]; h[h0 + 1] = psi[p0 + 1] + s * psi[p2];
            h[h1] = psi[p1] + s * psi[p3 + 1]; h[h1 + 1] = psi[p1 + 1] - s * psi[p3];
        } else {
            h[h0] = psi[p0] + s * psi[p2]; h[h0 + 1] = psi[p0 + 1] + s * psi[p2 + 1];
            h[h1] = psi[p1] + s * psi[p3]; h[h1 + 1] = psi[p1 + 1] + s * psi[p3 + 1];
        }
    }
}

template <typename R, int MU>
__device__ __forceinline__ void spin_recon_acc_s(const R (&g)[12], R s, R (&acc)[24]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int g0 = 2 * c, g1 = 6 + 2 * c;
        const int a0 = 2 * c, a1 = 6 + 2 * c, a2 = 12 + 2 * c, a3 = 18 + 2 * c;
        acc[a0] += g[g0]; acc[a0 + 1] += g[g0 + 1];
        acc[a1] += g[g1]; acc[a1 + 1] += g[g1 + 1];
        if (MU == 0) {
            acc[a2] += s * g[g1 + 1]; acc[a2 + 1] -= s * g[g1];
            acc[a3] += s * g[g0 + 1]; acc[a3 + 1] -= s * g[g0];
        } else if (MU == 1) {
            acc[a2] += s * g[g1]; acc[a2 + 1] += s * g[g1 + 1];
            acc[a3] -= s * g[g0]; acc[a3 + 1] -= s * g[g0 + 1];
        } else if (MU == 2) {
            acc[a2] += s * g[g0 + 1]; acc[a2 + 1] -= s * g[g0];
            acc[a3] -= s * g[g1 + 1]; acc[a3 + 1] += s * g[g1];
        } else {
            acc[a2] += s * g[g0]; acc[a2 + 1] += s * g[g0 + 1];
            acc[a3] += s * g[g1]; acc[a3 + 1] += s * g[g1 + 1];
        }
    }
}

__device__ __forceinline__ float shfl_xor16(float v) { return __shfl_xor_sync(0xffffffffu, v, 16); }
__device__ __forceinline__ double shfl_xor16(double v) { return __shfl_xor_sync(0xffffffffu, v, 16); }

struct PipeArgs {
    Geom g;
    const void* in;
    void* out;
    const void* W;
    const uint16_t* nbslot;     // [8][TS]      (this output parity)
    const int16_t* slot_dir;    // [NSLOT]
    const uint16_t* slot_lane;  // [NSLOT]
    int out_parity;
    int dagger;
};

template <typename R, int TPS, int NG, int TS, int NSLOT, int NST>
__global__ void __launch_bounds__(TS* TPS) dhop_pipe_kernel(const PipeArgs a) {
    using V = typename VT<R>::V;
    constexpr int K = VT<R>::K, VW = VT<R>::VW;
    constexpr int KG = (NG + VW - 1) / VW;
    constexpr int LPT = 8 / TPS;
    constexpr int NTHR = TS * TPS;
    constexpr int NLD = (NSLOT + NTHR - 1) / NTHR;
    constexpr int STAGE = K * NSLOT;   // vectors per stage

    extern __shared__ __align__(16) unsigned char smem_raw[];
    V* const stage0 = reinterpret_cast<V*>(smem_raw);

    const Geom& g = a.g;
    const int Ls = g.Ls;
    const int tile = blockIdx.x;
    const int tid = threadIdx.x;
    int sub, lane;
    if (TPS == 1) { sub = 0; lane = tid; }
    else { sub = (tid >> 4) & 1; lane = ((tid >> 5) << 4) + (tid & 15); }

    // tile coordinates and the 8 neighbouring tiles (periodic)
    int tc[4];
    tile_coords(g, tile, tc);

    // ---- loader set-up: source offsets (vector units, s = 0, k = 0) of this thread's stage slots
    const V* __restrict__ in = reinterpret_cast<const V*>(a.in);
    unsigned srcoff[NLD];
#pragma unroll
    for (int j = 0; j < NLD; ++j) {
        const int slot = tid + j * NTHR;
        srcoff[j] = 0;
        if (slot < NSLOT) {
            const int d = a.slot_dir[slot];
            int t2 = tile;
            if (d >= 0) {
                int nc[4] = {tc[0], tc[1], tc[2], tc[3]};
                const int mu = d >> 1;
                nc[mu] += (d & 1) ? -1 : +1;
                if (nc[mu] < 0) nc[mu] = g.NT[mu] - 1;
                if (nc[mu] >= g.NT[mu]) nc[mu] = 0;
                t2 = tile_index(g, nc);
            }
            srcoff[j] = (unsigned)t2 * (unsigned)(Ls * K * TS) + (unsigned)a.slot_lane[slot];
        }
    }
    auto issue = [&](int s, int st) {
        V* sp = stage0 + st * STAGE;
#pragma unroll
        for (int j = 0; j < NLD; ++j) {
            const int slot = tid + j * NTHR;
            if (NSLOT % NTHR == 0 || j + 1 < NLD || slot < NSLOT) {
                const V* src = in + srcoff[j] + (size_t)s * (K * TS);
#pragma unroll
                for (int k = 0; k < K; ++k) cp_async16(sp + k * NSLOT + slot, src + k * TS);
            }
        }
    };
    // ---- start the ring
#pragma unroll
    for (int s = 0; s < NST - 1; ++s) {
        if (s < Ls) issue(s, s);
        cp_async_commit();
    }

    // ---- links to registers (once per tile): rows 0,1 (+ row 2 rebuilt), antiperiodic sign folded in
    const int tt = lane / (TS / g.T[3]);
    const int tglob = tc[3] * g.T[3] + tt;
    R u[LPT][18];
    int myslot[LPT];
    {
        const V* __restrict__ Wt = reinterpret_cast<const V*>(a.W) + (size_t)tile * 8 * KG * TS + lane;
#pragma unroll
        for (int j = 0; j < LPT; ++j) {
            const int leg = (TPS == 1) ? j : 2 * j + sub;
            load_link<R, NG>(Wt + (size_t)leg * KG * TS, TS, u[j]);
            myslot[j] = a.nbslot[leg * TS + lane];
            const int mu = (TPS == 1) ? (j >> 1) : j;
            if (mu == 3 && g.antiperiodic_t) {
                const int dir = (TPS == 1) ? (j & 1) : sub;
                const bool flip = dir ? (tglob == 0) : (tglob == g.L[3] - 1);
                if (flip) {
#pragma unroll
                    for (int i = 0; i < 18; ++i) u[j][i] = -u[j][i];
                }
            }
        }
    }
    const R dsgn = a.dagger ? (R)-1 : (R)1;

    V* __restrict__ outp = reinterpret_cast<V*>(a.out) + (size_t)tile * Ls * K * TS + lane;
    int st = 0, st_issue = NST - 1;
    for (int s = 0; s < Ls; ++s) {
        cp_async_wait<NST - 2>();
        __syncthreads();
        if (s + NST - 1 < Ls) issue(s + NST - 1, st_issue);
        cp_async_commit();
        const V* sp = stage0 + st * STAGE;
        R acc[24];
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = (R)0;
#pragma unroll
        for (int j = 0; j < LPT; ++j) {
            const int mu = (TPS == 1) ? (j >> 1) : j;
            const int dir = (TPS == 1) ? (j & 1) : sub;
            const R sg = (dir ? (R)1 : (R)-1) * dsgn;     // forward leg: (1 - gamma), backward: (1 + gamma)
            R psi[24], h[12], gg[12];
            const V* p = sp + myslot[j];
#pragma unroll
            for (int k = 0; k < K; ++k) unpackv(p[k * NSLOT], psi + k * VW);
            if (mu == 0) { spin_project_s<R, 0>(psi, sg, h); su3_mul<R>(u[j], h, gg); spin_recon_acc_s<R, 0>(gg, sg, acc); }
            else if (mu == 1) { spin_project_s<R, 1>(psi, sg, h); su3_mul<R>(u[j], h, gg); spin_recon_acc_s<R, 1>(gg, sg, acc); }
            else if (mu == 2) { spin_project_s<R, 2>(psi, sg, h); su3_mul<R>(u[j], h, gg); spin_recon_acc_s<R, 2>(gg, sg, acc); }
            else { spin_project_s<R, 3>(psi, sg, h); su3_mul<R>(u[j], h, gg); spin_recon_acc_s<R, 3>(gg, sg, acc); }
        }
        V* o = outp + (size_t)s * (K * TS);
        if (TPS == 1) {
#pragma unroll
            for (int k = 0; k < K; ++k) o[k * TS] = packv(acc + k * VW);
        } else {
            // lane pair (l, l^16): each keeps one half of the 24 sums, sends the other half
            R mine[12];
#pragma unroll
            for (int i = 0; i < 12; ++i) {
                const R send = sub ? acc[i] : acc[12 + i];
                const R keep = sub ? acc[12 + i] : acc[i];
                mine[i] = keep + shfl_xor16(send);
            }
            V* o2 = o + (sub ? (K / 2) * TS : 0);
#pragma unroll
            for (int k = 0; k < K / 2; ++k) o2[k * TS] = packv(mine + k * VW);
        }
        st = (st + 1 == NST) ? 0 : st + 1;
        st_issue = (st_issue + 1 == NST) ? 0 : st_issue + 1;
    }
}

// ------------------------------------------------------------------------------------------ launch
template <typename R, int TPS, int NG, int TS, int NSLOT, int NST>
static dwf_status launch_pipe_t(dwf_ctx* c, const PipeArgs& a) {
    using V = typename VT<R>::V;
    constexpr int K = VT<R>::K;
    const size_t smem = (size_t)NST * K * NSLOT * sizeof(V);
    auto kern = dhop_pipe_kernel<R, TPS, NG, TS, NSLOT, NST>;
    static unsigned long long attr_done = 0;      // per device (dwf_internal.h)
    if (attr_needed(attr_done, c->device))
        DWF_CUDA_CHECK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<c->g.ntiles, TS * TPS, smem, c->stream>>>(a);
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

template <typename R, int TPS, int TS, int NSLOT, int NST>
static dwf_status launch_pipe_ng(dwf_ctx* c, const PipeArgs& a) {
    return c->compress12 ? launch_pipe_t<R, TPS, 12, TS, NSLOT, NST>(c, a) : launch_pipe_t<R, TPS, 18, TS, NSLOT, NST>(c, a);
}

// returns DWF_OK and sets *handled = true when a pipelined instantiation exists for this tile shape
dwf_status launch_dhop_pipe(dwf_ctx* c, void* out, const void* in, int out_parity, int dagger, int prec, bool* handled) {
    *handled = false;
    const int pr = (prec == DWF_F64) ? 1 : 0;
    if (!c->pipe_nbslot[pr] || c->g.Ls < 1) return DWF_OK;
    const Geom g = geom_prec(c, prec, c->nrhs_cur);
    PipeArgs a;
    a.g = g; a.in = in; a.out = out;
    a.W = (prec == DWF_F64) ? c->W64[out_parity] : c->W32[out_parity];
    a.nbslot = c->pipe_nbslot[pr] + (size_t)out_parity * 8 * g.TS;
    a.slot_dir = c->pipe_slot_dir[pr] + (size_t)out_parity * c->pipe_nslot;
    a.slot_lane = c->pipe_slot_lane[pr] + (size_t)out_parity * c->pipe_nslot;
    a.out_parity = out_parity; a.dagger = dagger;
    const int TS = g.TS, NS = c->pipe_nslot;
#define DWF_PIPE_CASE(TSV, NSV)                                                                          \
    if (TS == TSV && NS == NSV) {                                                                        \
        *handled = true;                                                                                 \
        if (prec == DWF_F64) return launch_pipe_ng<double, 2, TSV, NSV, (3 * 12 * NSV * 16 <= 232448 ? 3 : 2)>(c, a); \
        return launch_pipe_ng<float, 1, TSV, NSV, 3>(c, a);                                              \
    }
    DWF_PIPE_CASE(128, 384)   // 4x4x4x4
    DWF_PIPE_CASE(128, 416)   // 8x4x4x2 and permutations
    DWF_PIPE_CASE(64, 224)    // 4x4x4x2 and permutations
#undef DWF_PIPE_CASE
    return DWF_OK;
}

}  // namespace dwf
