// Site-local 5-D operators (readings C4, C5): every one of them acts on each (spin, colour) component
// separately with a real Ls x Ls matrix that depends only on the chirality of the component:
//     out_s = sum_s' T+[s][s'] in_s'   on P+ components (spin 0,1)
//     out_s = sum_s' T-[s][s'] in_s'   on P- components (spin 2,3)
// A = b5 + c5 Q, Mooee = bee - cee Q, Mooee^-1 (closed form), their adjoints and the products the
// Schur operator needs are all just different tables, built on the host in fp64.
// One thread owns one 16-byte vector (2 or 4 reals of one chirality) of one 4-D site and holds its
// whole Ls column in registers; loads and stores are coalesced over the lanes of a tile.
#include <cmath>
#include <cstring>

#include "dwf_layout.cuh"

namespace dwf {

// ------------------------------------------------------------------ host: coefficient tables
static void mat_zero(double* a) { memset(a, 0, sizeof(double) * 32 * 32); }
static void mat_mul(const double* a, const double* b, double* c, int n) {  // c = a b   (32-stride)
    double t[32 * 32];
    mat_zero(t);
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            double s = 0;
            for (int k = 0; k < n; ++k) s += a[i * 32 + k] * b[k * 32 + j];
            t[i * 32 + j] = s;
        }
    memcpy(c, t, sizeof(t));
}

void build_tables(dwf_ctx* c) {
    const int Ls = c->g.Ls;
    const double bee = 1.0 + c->b5 * (4.0 - c->M5), cee = 1.0 - c->c5 * (4.0 - c->M5);
    const double mf = c->mf;
    // s-shifts with the -mf walls: (S_dn psi)_s = psi_{s-1}, (S_up psi)_s = psi_{s+1}
    double up[32 * 32], dn[32 * 32], id[32 * 32];
    mat_zero(up); mat_zero(dn); mat_zero(id);
    for (int s = 0; s < Ls; ++s) {
        id[s * 32 + s] = 1.0;
        if (s + 1 < Ls) up[s * 32 + s + 1] += 1.0; else up[s * 32 + 0] += -mf;
        if (s - 1 >= 0) dn[s * 32 + s - 1] += 1.0; else dn[s * 32 + Ls - 1] += -mf;
    }
    auto lin = [&](double a, double b, const double* S, double* out) {   // out = a*1 + b*S
        for (int i = 0; i < 32 * 32; ++i) out[i] = a * id[i] + b * S[i];
    };
    // Q = P- S_up + P+ S_dn  ->  P+ components see S_dn, P- components see S_up;  Q^dag swaps them
    lin(c->b5, c->c5, dn, c->tab[OP_A].p);      lin(c->b5, c->c5, up, c->tab[OP_A].m);
    lin(c->b5, c->c5, up, c->tab[OP_ADAG].p);   lin(c->b5, c->c5, dn, c->tab[OP_ADAG].m);
    lin(bee, -cee, dn, c->tab[OP_MEE].p);       lin(bee, -cee, up, c->tab[OP_MEE].m);
    lin(bee, -cee, up, c->tab[OP_MEEDAG].p);    lin(bee, -cee, dn, c->tab[OP_MEEDAG].m);
    // closed-form inverse (reading C5): r = cee/bee, d = bee (1 + mf r^Ls)
    const double r = cee / bee, d = bee * (1.0 + mf * std::pow(r, Ls));
    double* ip = c->tab[OP_MEEINV].p; double* im = c->tab[OP_MEEINV].m;
    mat_zero(ip); mat_zero(im);
    for (int s = 0; s < Ls; ++s)
        for (int t = 0; t < Ls; ++t) {
            ip[s * 32 + t] = std::pow(r, ((s - t) % Ls + Ls) % Ls) * (s >= t ? 1.0 : -mf) / d;
            im[s * 32 + t] = std::pow(r, ((t - s) % Ls + Ls) % Ls) * (t >= s ? 1.0 : -mf) / d;
        }
    memcpy(c->tab[OP_MEEINVDAG].p, im, sizeof(double) * 32 * 32);
    memcpy(c->tab[OP_MEEINVDAG].m, ip, sizeof(double) * 32 * 32);
    mat_mul(c->tab[OP_A].p, c->tab[OP_MEEINV].p, c->tab[OP_A_MEEINV].p, Ls);
    mat_mul(c->tab[OP_A].m, c->tab[OP_MEEINV].m, c->tab[OP_A_MEEINV].m, Ls);
    mat_mul(c->tab[OP_MEEINVDAG].p, c->tab[OP_ADAG].p, c->tab[OP_MEEINVDAG_ADAG].p, Ls);
    mat_mul(c->tab[OP_MEEINVDAG].m, c->tab[OP_ADAG].m, c->tab[OP_MEEINVDAG_ADAG].m, Ls);
}

// ------------------------------------------------------------------ device
template <typename R> struct V5;
template <> struct V5<float> { using V = float4; static constexpr int VW = 4, K = 6; };
template <> struct V5<double> { using V = double2; static constexpr int VW = 2, K = 12; };

__device__ __forceinline__ void fmav(float4& a, float t, const float4& x) {
    a.x = fmaf(t, x.x, a.x); a.y = fmaf(t, x.y, a.y); a.z = fmaf(t, x.z, a.z); a.w = fmaf(t, x.w, a.w);
}
__device__ __forceinline__ void fmav(double2& a, double t, const double2& x) {
    a.x = fma(t, x.x, a.x); a.y = fma(t, x.y, a.y);
}
__device__ __forceinline__ void scalev(float4& a, float t) { a.x *= t; a.y *= t; a.z *= t; a.w *= t; }
__device__ __forceinline__ void scalev(double2& a, double t) { a.x *= t; a.y *= t; }
__device__ __forceinline__ float4 zerov(float4*) { return make_float4(0.f, 0.f, 0.f, 0.f); }
__device__ __forceinline__ double2 zerov(double2*) { return make_double2(0.0, 0.0); }
__device__ __forceinline__ double norm2v(const float4& a) {
    return (double)a.x * a.x + (double)a.y * a.y + (double)a.z * a.z + (double)a.w * a.w;
}
__device__ __forceinline__ double norm2v(const double2& a) { return a.x * a.x + a.y * a.y; }

__device__ __forceinline__ double block_reduce_sum(double v) {
    __shared__ double wsum[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) wsum[w] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    v = (threadIdx.x < nw) ? wsum[threadIdx.x] : 0.0;
    if (w == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    }
    return v;   // valid in thread 0
}

// mode 0: out = T1 x ; mode 1: out = T1 x + yscale*y ; mode 2: out = T1 x + yscale * T2 y
// tables in global memory: [chirality][Ls*Ls] of R, row-major s, s'
template <typename R, int LS>
__global__ void __launch_bounds__(128) op5_kernel(int Ls_rt, int TS, unsigned nvec_site /* Vh*K */,
                                                  const typename V5<R>::V* __restrict__ x,
                                                  const typename V5<R>::V* __restrict__ y,
                                                  typename V5<R>::V* __restrict__ out, const R* __restrict__ T1,
                                                  const R* __restrict__ T2, R yscale, int mode,
                                                  double* __restrict__ partials) {
    using V = typename V5<R>::V;
    constexpr int K = V5<R>::K;
    const int Ls = (LS > 0) ? LS : Ls_rt;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    R* sT1 = reinterpret_cast<R*>(smem_raw);          // [2][Ls*Ls]
    R* sT2 = sT1 + 2 * Ls * Ls;
    for (int i = threadIdx.x; i < 2 * Ls * Ls; i += blockDim.x) {
        sT1[i] = T1[i];
        if (mode == 2) sT2[i] = T2[i];
    }
    __syncthreads();
    const unsigned gid = blockIdx.x * blockDim.x + threadIdx.x;
    double nrm = 0.0;
    if (gid < nvec_site) {
        const unsigned per_tile = (unsigned)K * TS;
        const unsigned tile = gid / per_tile, j = gid - tile * per_tile;
        const int k = j / TS;
        const int chir = (k < K / 2) ? 0 : 1;
        const size_t base = ((size_t)tile * gridDim.y + blockIdx.y) * Ls * per_tile + j;     // blockIdx.y: right-hand side
        const R* t1 = sT1 + chir * Ls * Ls;
        const R* t2 = sT2 + chir * Ls * Ls;
        if (LS > 0) {
            V xin[LS > 0 ? LS : 1];
#pragma unroll
            for (int s = 0; s < LS; ++s) xin[s] = x[base + (size_t)s * per_tile];
            V yin[LS > 0 ? LS : 1];
            if (mode == 2) {
#pragma unroll
                for (int s = 0; s < LS; ++s) yin[s] = y[base + (size_t)s * per_tile];
            }
#pragma unroll
            for (int s = 0; s < LS; ++s) {
                V acc = zerov((V*)nullptr);
#pragma unroll
                for (int sp = 0; sp < LS; ++sp) fmav(acc, t1[s * LS + sp], xin[sp]);
                if (mode == 1) {
                    fmav(acc, yscale, y[base + (size_t)s * per_tile]);
                } else if (mode == 2) {
                    V a2 = zerov((V*)nullptr);
#pragma unroll
                    for (int sp = 0; sp < LS; ++sp) fmav(a2, t2[s * LS + sp], yin[sp]);
                    fmav(acc, yscale, a2);
                }
                out[base + (size_t)s * per_tile] = acc;
                nrm += norm2v(acc);
            }
        } else {
            // generic Ls: re-read the column per output slice (L1-resident); out must not alias x or y
            for (int s = 0; s < Ls; ++s) {
                V acc = zerov((V*)nullptr);
                for (int sp = 0; sp < Ls; ++sp) fmav(acc, t1[s * Ls + sp], x[base + (size_t)sp * per_tile]);
                if (mode == 1) {
                    fmav(acc, yscale, y[base + (size_t)s * per_tile]);
                } else if (mode == 2) {
                    V a2 = zerov((V*)nullptr);
                    for (int sp = 0; sp < Ls; ++sp) fmav(a2, t2[s * Ls + sp], y[base + (size_t)sp * per_tile]);
                    fmav(acc, yscale, a2);
                }
                out[base + (size_t)s * per_tile] = acc;
                nrm += norm2v(acc);
            }
        }
    }
    if (partials != nullptr) {
        double tot = block_reduce_sum(nrm);
        if (threadIdx.x == 0) partials[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = tot;
    }
}


// CG vector step fused with the next A p (fused CG loop, dwf_api.cu):  x += alpha p;  p <- r + beta p;  ap = A p,
// A = b5 + c5 Q (reading C5).  One thread owns one 16-byte vector column of one 4-D site and walks it in sweep order
// (s ascending on P+ components, descending on P-), so (Q p)_j is the previous element, the -mf wall at j = 0.
// init: p <- r, ap = A p, x untouched.  alpha = sc[slot_c]/sc[slot_d], beta = sc[slot_cn]/sc[slot_c] of the thread's
// right-hand side (blockIdx.y).  A system whose stopping test fired at an EARLIER iteration (conv[rhs] in [0, iter)) is
// frozen: the host runs one iteration ahead of the residuals it has read, and other systems of a batch may still iterate.
// A frozen system keeps x and p; its ap is set to zero (see below) and cg_r_kernel leaves its r alone.
template <typename R>
__global__ void __launch_bounds__(128) cg_xp_kernel(int Ls, int TS, unsigned nvec_site, typename V5<R>::V* __restrict__ x,
                                                    typename V5<R>::V* __restrict__ p,
                                                    const typename V5<R>::V* __restrict__ r,
                                                    typename V5<R>::V* __restrict__ ap, const double* __restrict__ sc,
                                                    int slot_c, int slot_d, int slot_cn, int init, R b5, R c5, R mf,
                                                    const int* __restrict__ conv, int iter) {
    using V = typename V5<R>::V;
    constexpr int K = V5<R>::K;
    const unsigned gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= nvec_site) return;
    const int rhs = blockIdx.y;
    const unsigned per_tile = (unsigned)K * TS;
    const unsigned tile = gid / per_tile, j = gid - tile * per_tile;
    const int k = j / TS;
    const bool rev = (k >= K / 2);
    const size_t base = ((size_t)tile * gridDim.y + rhs) * Ls * per_tile + j;
    if (!init) {
        const int cv = conv[rhs];
        if (cv >= 0 && cv < iter) {
            // frozen: x and p stay.  ap is the buffer the Dhop chain works in, so it holds that chain's last output, not
            // A p: zero it, the chain of this system then carries zeros (and cg_r skips the system) instead of feeding
            // its own output back into itself iteration after iteration until it overflows.
            for (int jj = 0; jj < Ls; ++jj) ap[base + (size_t)jj * per_tile] = zerov((V*)nullptr);
            return;
        }
    }
    R alpha = (R)0, beta = (R)0;
    if (!init) {
        const double cc = sc[slot_c * MAXR + rhs];
        alpha = (R)(cc / sc[slot_d * MAXR + rhs]);
        beta = (R)(sc[slot_cn * MAXR + rhs] / cc);
    }
    const size_t olast = base + (size_t)(rev ? 0 : Ls - 1) * per_tile;
    V prev = r[olast];
    if (!init) fmav(prev, beta, p[olast]);
    scalev(prev, -mf);
#pragma unroll 4
    for (int jj = 0; jj < Ls; ++jj) {
        const size_t o = base + (size_t)(rev ? Ls - 1 - jj : jj) * per_tile;
        V pn = r[o];
        if (!init) {
            const V pv = p[o];
            V xv = x[o];
            fmav(xv, alpha, pv);
            x[o] = xv;
            fmav(pn, beta, pv);
        }
        p[o] = pn;
        V a = zerov((V*)nullptr);
        fmav(a, b5, pn);
        fmav(a, c5, prev);
        ap[o] = a;
        prev = pn;
    }
}

dwf_status launch_cg_xp(dwf_ctx* c, void* x, void* p, const void* r, void* ap, int prec, int slot_c, int slot_d,
                        int slot_cn, int init, int iter) {
    const Geom& g = c->g;
    const int block = 128;
    if (prec == DWF_F64) {
        const unsigned nvec_site = (unsigned)g.Vh * 12;
        const dim3 grid((nvec_site + block - 1) / block, c->nrhs_cur);
        cg_xp_kernel<double><<<grid, block, 0, c->stream>>>(
            g.Ls, g.TS, nvec_site, (double2*)x, (double2*)p, (const double2*)r, (double2*)ap, c->scalars, slot_c, slot_d,
            slot_cn, init, c->b5, c->c5, c->mf, c->cg_conv, iter);
    } else {
        const unsigned nvec_site = (unsigned)g.Vh * 6;
        const dim3 grid((nvec_site + block - 1) / block, c->nrhs_cur);
        cg_xp_kernel<float><<<grid, block, 0, c->stream>>>(
            g.Ls, g.TS, nvec_site, (float4*)x, (float4*)p, (const float4*)r, (float4*)ap, c->scalars, slot_c, slot_d,
            slot_cn, init, (float)c->b5, (float)c->c5, (float)c->mf, c->cg_conv, iter);
    }
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

// fixed-tree final reduction of the per-block partials into one device scalar per right-hand side (block = rhs):
// partials[rhs * n + i] -> result[rhs].  With `target` set it is also the CG's stopping test (reading C8), kept on the
// device: the first iteration at which |r|^2 <= target[rhs] is recorded in conv[rhs].
__global__ void __launch_bounds__(1024) reduce_partials_kernel(const double* __restrict__ partials, int n,
                                                               double* __restrict__ result, const double* __restrict__ target,
                                                               int* __restrict__ conv, int iter) {
    const int rhs = blockIdx.x;
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += 1024) v += partials[(size_t)rhs * n + i];
    double tot = block_reduce_sum(v);
    if (threadIdx.x == 0) {
        result[rhs] = tot;
        if (target != nullptr && conv[rhs] < 0 && tot <= target[rhs]) conv[rhs] = iter;
    }
}

dwf_status ensure_partials(dwf_ctx* c, int n) {
    n *= c->nrhs_cur;
    if (n <= c->npartials) return DWF_OK;
    if (c->partials) cudaFree(c->partials);
    c->partials = nullptr;
    c->npartials = 0;
    if (cudaMalloc(&c->partials, sizeof(double) * (size_t)n) != cudaSuccess) {
        c->err = "cudaMalloc(partials) failed";
        return DWF_ENOMEM;
    }
    c->npartials = n;
    return DWF_OK;
}

// n partials per right-hand side -> scalars[slot][rhs]; iter > 0: also the stopping test of CG iteration `iter`
dwf_status launch_reduce(dwf_ctx* c, int n, int slot, int iter) {
    reduce_partials_kernel<<<c->nrhs_cur, 1024, 0, c->stream>>>(c->partials, n, c->scalars + (size_t)slot * MAXR,
                                                                iter > 0 ? c->cg_target : nullptr, c->cg_conv, iter);
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

template <typename R>
static dwf_status launch_op5_t(dwf_ctx* c, void* out, const void* x, int op1, const void* y, int op2, double yscale,
                               int mode, int norm_slot) {
    using V = typename V5<R>::V;
    constexpr int K = V5<R>::K;
    const Geom& g = c->g;
    const int Ls = g.Ls;
    const unsigned nvec_site = (unsigned)g.Vh * K;
    const int block = 128;
    const int gridx = (int)((nvec_site + block - 1) / block);
    const dim3 grid(gridx, c->nrhs_cur);
    const R* tabs = (sizeof(R) == 8) ? (const R*)c->dtab.d64 : (const R*)c->dtab.d32;
    const R* T1 = tabs + (size_t)op1 * 2 * Ls * Ls;
    const R* T2 = (mode == 2) ? tabs + (size_t)op2 * 2 * Ls * Ls : nullptr;
    double* partials = nullptr;
    if (norm_slot >= 0) {
        dwf_status st = ensure_partials(c, gridx);
        if (st != DWF_OK) return st;
        partials = c->partials;
    }
    const size_t smem = sizeof(R) * 4 * Ls * Ls;
#define DWF_OP5_LAUNCH(LSV)                                                                                  \
    op5_kernel<R, LSV><<<grid, block, smem, c->stream>>>(Ls, g.TS, nvec_site, (const V*)x, (const V*)y, (V*)out, T1, \
                                                         T2, (R)yscale, mode, partials)
    switch (Ls) {
        case 4: DWF_OP5_LAUNCH(4); break;
        case 8: DWF_OP5_LAUNCH(8); break;
        case 12: DWF_OP5_LAUNCH(12); break;
        case 16: DWF_OP5_LAUNCH(16); break;
        default:
            if (out == x || out == y) { c->err = "op5: generic-Ls path cannot run in place"; return DWF_EINVAL; }
            DWF_OP5_LAUNCH(0);
            break;
    }
#undef DWF_OP5_LAUNCH
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    if (norm_slot >= 0) return launch_reduce(c, gridx, norm_slot, 0);
    return DWF_OK;
}

// out = T[op1] x (+ yscale*y | + yscale*T[op2] y);  y == nullptr: mode 0; op2 < 0: mode 1; else mode 2.
// norm_slot >= 0: |out|^2 is reduced into c->scalars[norm_slot].
dwf_status launch_op5(dwf_ctx* c, void* out, const void* x, int op1, const void* y, int op2, double yscale, int prec,
                      int norm_slot) {
    const int mode = (y == nullptr) ? 0 : (op2 < 0 ? 1 : 2);
    if (prec == DWF_F64) return launch_op5_t<double>(c, out, x, op1, y, op2, yscale, mode, norm_slot);
    return launch_op5_t<float>(c, out, x, op1, y, op2, yscale, mode, norm_slot);
}

}  // namespace dwf

namespace dwf {
// CG residual step (reading C8: r -= alpha Mpc^dag q) in one streaming column kernel.  The last step of Mpc^dag,
// z = Mee^dag q - 1/4 A^dag d, is bidiagonal in s on both operands (reading C5): in sweep order (daggered operators:
// s descending on P+ components, ascending on P-) (Q^dag x)_j is the previous element, the -mf wall at j = 0, so
//     z_j = bee q_j - cee q_{j-1} + yscale (b5 d_j + c5 d_{j-1})
// is formed in registers and never stored; r -= alpha z with alpha = sc[slot_c]/sc[slot_d]; |r|^2 -> partials.
template <typename R>
__global__ void __launch_bounds__(128) cg_r_kernel(int Ls, int TS, unsigned nvec_site, typename V5<R>::V* __restrict__ r,
                                                   const typename V5<R>::V* __restrict__ q,
                                                   const typename V5<R>::V* __restrict__ d, const double* __restrict__ sc,
                                                   int slot_c, int slot_d, R bee, R mcee, R yb5, R yc5, R mf,
                                                   double* __restrict__ partials, const int* __restrict__ conv, int iter) {
    using V = typename V5<R>::V;
    constexpr int K = V5<R>::K;
    const unsigned gid = blockIdx.x * blockDim.x + threadIdx.x;
    double nrm = 0.0;
    // a system whose stopping test fired at an earlier iteration is frozen (cg_xp_kernel): its chain carries zeros, its
    // scalars are no longer meaningful (d = 0), r stays as it is and the partial written for it is 0
    const int cv = conv[blockIdx.y];
    const bool frozen = (cv >= 0 && cv < iter);
    if (gid < nvec_site && !frozen) {
        const unsigned per_tile = (unsigned)K * TS;
        const unsigned tile = gid / per_tile, j = gid - tile * per_tile;
        const int k = j / TS;
        const bool rev = (k < K / 2);          // daggered: P+ components walk s downwards
        const size_t base = ((size_t)tile * gridDim.y + blockIdx.y) * Ls * per_tile + j;     // blockIdx.y: right-hand side
        const R alpha = (R)(sc[slot_c * MAXR + blockIdx.y] / sc[slot_d * MAXR + blockIdx.y]);
        const size_t olast = base + (size_t)(rev ? 0 : Ls - 1) * per_tile;
        V qprev = q[olast], dprev = d[olast];
        scalev(qprev, -mf);
        scalev(dprev, -mf);
#pragma unroll 4
        for (int jj = 0; jj < Ls; ++jj) {
            const size_t o = base + (size_t)(rev ? Ls - 1 - jj : jj) * per_tile;
            const V qv = q[o], dv = d[o];
            V z = zerov((V*)nullptr);
            fmav(z, bee, qv);
            fmav(z, mcee, qprev);
            fmav(z, yb5, dv);
            fmav(z, yc5, dprev);
            V rv = r[o];
            fmav(rv, -alpha, z);
            r[o] = rv;
            nrm += norm2v(rv);
            qprev = qv;
            dprev = dv;
        }
    }
    const double tot = block_reduce_sum(nrm);
    if (threadIdx.x == 0) partials[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = tot;
}

dwf_status launch_cg_r(dwf_ctx* c, void* r, const void* q, const void* d, double yscale, int prec, int slot_c, int slot_d,
                       int norm_slot, int iter) {
    const Geom& g = c->g;
    const double bee = 1.0 + c->b5 * (4.0 - c->M5), cee = 1.0 - c->c5 * (4.0 - c->M5);
    const int block = 128;
    const unsigned nvec_site = (unsigned)g.Vh * (prec == DWF_F64 ? 12 : 6);
    const int gridx = (int)((nvec_site + block - 1) / block);
    const dim3 grid(gridx, c->nrhs_cur);
    dwf_status st = ensure_partials(c, gridx);
    if (st != DWF_OK) return st;
    if (prec == DWF_F64)
        cg_r_kernel<double><<<grid, block, 0, c->stream>>>(g.Ls, g.TS, nvec_site, (double2*)r, (const double2*)q,
                                                           (const double2*)d, c->scalars, slot_c, slot_d, bee, -cee,
                                                           yscale * c->b5, yscale * c->c5, c->mf, c->partials, c->cg_conv, iter);
    else
        cg_r_kernel<float><<<grid, block, 0, c->stream>>>(g.Ls, g.TS, nvec_site, (float4*)r, (const float4*)q,
                                                          (const float4*)d, c->scalars, slot_c, slot_d, (float)bee,
                                                          (float)-cee, (float)(yscale * c->b5), (float)(yscale * c->c5),
                                                          (float)c->mf, c->partials, c->cg_conv, iter);
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return launch_reduce(c, gridx, norm_slot, iter);
}
}  // namespace dwf
