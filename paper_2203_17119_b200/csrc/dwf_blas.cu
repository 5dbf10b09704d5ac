// BLAS-1 kernels of the CG (reading C8): 128-bit grid-stride streaming with the norm fused into the
// update kernel; every reduction is accumulated in fp64 through warp shuffles -> one partial per block ->
// a fixed-tree single-block pass (deterministic: the same inputs always give the same bits).
// CG scalars stay on the device: alpha = c/d and beta = c'/c are formed inside the kernels from the
// scalar slots, so the host only reads one double per iteration for the stopping test.
#include "dwf_internal.h"

namespace dwf {

// Batched fields (dwf_internal.h): the kernels that need a per-system scalar run with blockIdx.y = right-hand side and map
// their running index i over ONE system's vectors to the batched field: i = tile * chunk + off -> (tile * N + rhs) * chunk + off,
// chunk = Ls * K * TS vectors (one tile of one system).  N = 1: the identity.
__device__ __forceinline__ size_t rhs_index(size_t i, unsigned chunk) {
    if (gridDim.y == 1) return i;
    const size_t tile = i / chunk;
    return (tile * gridDim.y + blockIdx.y) * chunk + (i - tile * chunk);
}

template <typename R> struct VB;
template <> struct VB<float> { using V = float4; static constexpr int VW = 4; };
template <> struct VB<double> { using V = double2; static constexpr int VW = 2; };

__device__ __forceinline__ double blk_sum(double v) {
    __shared__ double wsum[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) wsum[w] = v;
    __syncthreads();
    const int nw = (blockDim.x + 31) >> 5;
    v = (threadIdx.x < nw) ? wsum[threadIdx.x] : 0.0;
    if (w == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    }
    return v;
}

__device__ __forceinline__ double n2(const float4& a) {
    return (double)a.x * a.x + (double)a.y * a.y + (double)a.z * a.z + (double)a.w * a.w;
}
__device__ __forceinline__ double n2(const double2& a) { return a.x * a.x + a.y * a.y; }
__device__ __forceinline__ float4 axpyv(float a, const float4& x, const float4& y) {
    return make_float4(fmaf(a, x.x, y.x), fmaf(a, x.y, y.y), fmaf(a, x.z, y.z), fmaf(a, x.w, y.w));
}
__device__ __forceinline__ double2 axpyv(double a, const double2& x, const double2& y) {
    return make_double2(fma(a, x.x, y.x), fma(a, x.y, y.y));
}

template <typename R>
__global__ void __launch_bounds__(256) norm2_kernel(const typename VB<R>::V* __restrict__ v, size_t nvec, unsigned chunk,
                                                    double* __restrict__ partials) {
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x)
        acc += n2(v[rhs_index(i, chunk)]);
    double tot = blk_sum(acc);
    if (threadIdx.x == 0) partials[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = tot;
}

// x += a p ; r -= a z ; partial |r|^2 ;  a = sc[slot_c]/sc[slot_d]
template <typename R>
__global__ void __launch_bounds__(256) cg_update_kernel(typename VB<R>::V* __restrict__ x, typename VB<R>::V* __restrict__ r,
                                                        const typename VB<R>::V* __restrict__ p,
                                                        const typename VB<R>::V* __restrict__ z, size_t nvec, unsigned chunk,
                                                        const double* __restrict__ sc, int slot_c, int slot_d,
                                                        double* __restrict__ partials, const int* __restrict__ conv, int iter) {
    const int rhs = blockIdx.y;
    const R a = (R)(sc[slot_c * MAXR + rhs] / sc[slot_d * MAXR + rhs]);
    const int cv = conv[rhs];
    const bool frozen = (cv >= 0 && cv < iter);       // stopping test fired at an earlier iteration: x stays
    double acc = 0.0;
    for (size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < nvec; i0 += (size_t)gridDim.x * blockDim.x) {
        const size_t i = rhs_index(i0, chunk);
        if (!frozen) x[i] = axpyv(a, p[i], x[i]);
        typename VB<R>::V rn = axpyv(-a, z[i], r[i]);
        r[i] = rn;
        acc += n2(rn);
    }
    double tot = blk_sum(acc);
    if (threadIdx.x == 0) partials[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = tot;
}

// p = r + b p ; b = sc[slot_cn]/sc[slot_c]
template <typename R>
__global__ void __launch_bounds__(256) xpay_kernel(typename VB<R>::V* __restrict__ p, const typename VB<R>::V* __restrict__ r,
                                                   size_t nvec, unsigned chunk, const double* __restrict__ sc, int slot_cn,
                                                   int slot_c) {
    const R b = (R)(sc[slot_cn * MAXR + blockIdx.y] / sc[slot_c * MAXR + blockIdx.y]);
    for (size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < nvec; i0 += (size_t)gridDim.x * blockDim.x) {
        const size_t i = rhs_index(i0, chunk);
        p[i] = axpyv(b, p[i], r[i]);
    }
}

// y += a x
template <typename R>
__global__ void __launch_bounds__(256) axpy_kernel(typename VB<R>::V* __restrict__ y, const typename VB<R>::V* __restrict__ x,
                                                   R a, size_t nvec) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x)
        y[i] = axpyv(a, x[i], y[i]);
}

// out = a - b
template <typename R>
__global__ void __launch_bounds__(256) sub_kernel(typename VB<R>::V* __restrict__ out, const typename VB<R>::V* __restrict__ a,
                                                  const typename VB<R>::V* __restrict__ b, size_t nvec) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x)
        out[i] = axpyv((R)-1, b[i], a[i]);
}

// ---- multishift CG (dwf_multishift_cg): the scalar recurrences live on the device (MsState, one per context), so that the
// loop needs no host round trip: two one-thread kernels form alpha / zeta / the update coefficients from the reduction
// slots, the vector kernels read them from MsState.  The stopping test is the CG's (cg_conv[0], cg_target[0]).
// before the residual step: d = |q|^2 + s0 |p_0|^2, alpha = c / d, zeta_i', ax_i = alpha zeta_i' / zeta_i
__global__ void ms_alpha_kernel(MsState* __restrict__ st, const double* __restrict__ sc, int slot_d) {
    if (threadIdx.x != 0) return;
    const double d = sc[slot_d * MAXR] + st->s0 * st->p0n2;
    const double alpha = st->cc / d;
    st->alpha = alpha;
    for (int i = 0; i < st->n; ++i) {
        const double z = st->zeta[i], zo = st->zeta_old[i];
        const double zn = z * zo * st->alpha_old / (alpha * st->beta_old * (zo - z) + zo * st->alpha_old * (1.0 + st->delta[i] * alpha));
        st->znew[i] = zn;
        st->ax[i] = alpha * zn / z;
    }
}
// after the residual step: beta = c' / c, p_i = zeta_i' r + beta (zeta_i' / zeta_i)^2 p_i; then the state moves on
__global__ void ms_beta_kernel(MsState* __restrict__ st, const double* __restrict__ sc, int slot_cn) {
    if (threadIdx.x != 0) return;
    const double cn = sc[slot_cn * MAXR];
    const double beta = cn / st->cc;
    for (int i = 0; i < st->n; ++i) {
        const double ratio = st->znew[i] / st->zeta[i];
        st->zr[i] = st->znew[i];
        st->bp[i] = beta * ratio * ratio;
        st->zeta_old[i] = st->zeta[i];
        st->zeta[i] = st->znew[i];
    }
    st->alpha_old = st->alpha;
    st->beta_old = beta;
    st->cc = cn;
}
// |p_0|^2 of the new p_0 -> state (read by the next ms_alpha_kernel)
__global__ void ms_p0_kernel(MsState* __restrict__ st, const double* __restrict__ sc, int slot) {
    if (threadIdx.x == 0) st->p0n2 = sc[slot * MAXR];
}

// r -= alpha (z + s0 p_0) ; |r|^2
template <typename R>
__global__ void __launch_bounds__(256) ms_r_kernel(typename VB<R>::V* __restrict__ r, const typename VB<R>::V* __restrict__ z,
                                                   const typename VB<R>::V* __restrict__ p0, const MsState* __restrict__ st,
                                                   size_t nvec, double* __restrict__ partials) {
    const R a = (R)st->alpha, as0 = (R)(st->alpha * st->s0);
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        typename VB<R>::V v = axpyv(-a, z[i], r[i]);
        v = axpyv(-as0, p0[i], v);
        r[i] = v;
        acc += n2(v);
    }
    acc = blk_sum(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc;
}

// for every shift i: x_i += ax_i p_i ; p_i = zr_i r + bp_i p_i ; |p_0|^2 of the new p_0.  r is read once.  A system whose
// stopping test fired at an earlier iteration (conv[0] in [0, iter)) is left alone: the host runs one iteration ahead.
template <typename R>
__global__ void __launch_bounds__(256) ms_update_kernel(typename VB<R>::V* __restrict__ x, typename VB<R>::V* __restrict__ p,
                                                        const typename VB<R>::V* __restrict__ r, size_t nvec,
                                                        const MsState* __restrict__ st, double* __restrict__ partials,
                                                        const int* __restrict__ conv, int iter) {
    const int cv = conv[0];
    if (cv >= 0 && cv < iter) { if (threadIdx.x == 0) partials[blockIdx.x] = 0.0; return; }
    const int n = st->n;
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        const typename VB<R>::V rv = r[i];
        for (int k = 0; k < n; ++k) {
            const typename VB<R>::V pv = p[(size_t)k * nvec + i];
            x[(size_t)k * nvec + i] = axpyv((R)st->ax[k], pv, x[(size_t)k * nvec + i]);
            typename VB<R>::V pn = axpyv((R)st->bp[k], pv, typename VB<R>::V{});
            pn = axpyv((R)st->zr[k], rv, pn);
            p[(size_t)k * nvec + i] = pn;
            if (k == 0) acc += n2(pn);
        }
    }
    acc = blk_sum(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc;
}

// out = a x + b y + c z   (Chebyshev recurrence step; out may alias z)
template <typename R>
__global__ void __launch_bounds__(256) lincomb3_kernel(typename VB<R>::V* out, const typename VB<R>::V* __restrict__ x,
                                                       const typename VB<R>::V* __restrict__ y, const typename VB<R>::V* z, R a,
                                                       R b, R c, size_t nvec) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
        typename VB<R>::V v = axpyv(c, z[i], typename VB<R>::V{});
        v = axpyv(b, y[i], v);
        out[i] = axpyv(a, x[i], v);
    }
}

static inline int blas_grid(const dwf_ctx* c, size_t nvec) {
    size_t want = (nvec + 255) / 256;
    size_t cap = (size_t)c->num_sms * 8;     // 8 CTAs of 256 threads per SM, one wave
    return (int)(want < cap ? (want ? want : 1) : cap);
}

#define DWF_BLAS_DISPATCH(prec, CALL32, CALL64) \
    do { if ((prec) == DWF_F64) { CALL64; } else { CALL32; } } while (0)

// vectors of one tile of one system (the unit the batched layout interleaves)
static inline unsigned tile_chunk(const dwf_ctx* c, int prec) { return (unsigned)c->g.Ls * (prec == DWF_F64 ? 12 : 6) * c->g.TS; }

// nreal: reals of ONE system; with c->nrhs_cur > 1 the field is batched and every system gets its own norm
dwf_status launch_norm2(dwf_ctx* c, const void* v, int prec, size_t nreal, int slot) {
    const size_t nvec = nreal / (prec == DWF_F64 ? 2 : 4);
    const int gridx = blas_grid(c, nvec);
    const dim3 grid(gridx, c->nrhs_cur);
    const unsigned chunk = tile_chunk(c, prec);
    dwf_status st = ensure_partials(c, gridx);
    if (st != DWF_OK) return st;
    DWF_BLAS_DISPATCH(prec, (norm2_kernel<float><<<grid, 256, 0, c->stream>>>((const float4*)v, nvec, chunk, c->partials)),
                      (norm2_kernel<double><<<grid, 256, 0, c->stream>>>((const double2*)v, nvec, chunk, c->partials)));
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return launch_reduce(c, gridx, slot);
}

dwf_status launch_cg_update(dwf_ctx* c, void* x, void* r, const void* p, const void* z, int prec, size_t nreal,
                            int slot_c, int slot_d, int slot_cn, int iter) {
    const size_t nvec = nreal / (prec == DWF_F64 ? 2 : 4);
    const int gridx = blas_grid(c, nvec);
    const dim3 grid(gridx, c->nrhs_cur);
    const unsigned chunk = tile_chunk(c, prec);
    dwf_status st = ensure_partials(c, gridx);
    if (st != DWF_OK) return st;
    DWF_BLAS_DISPATCH(prec,
                      (cg_update_kernel<float><<<grid, 256, 0, c->stream>>>((float4*)x, (float4*)r, (const float4*)p,
                                                                          (const float4*)z, nvec, chunk, c->scalars, slot_c,
                                                                          slot_d, c->partials, c->cg_conv, iter)),
                      (cg_update_kernel<double><<<grid, 256, 0, c->stream>>>((double2*)x, (double2*)r, (const double2*)p,
                                                                           (const double2*)z, nvec, chunk, c->scalars, slot_c,
                                                                           slot_d, c->partials, c->cg_conv, iter)));
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return launch_reduce(c, gridx, slot_cn, iter);
}

dwf_status launch_xpay(dwf_ctx* c, void* p, const void* r, int prec, size_t nreal, int slot_cn, int slot_c) {
    const size_t nvec = nreal / (prec == DWF_F64 ? 2 : 4);
    const dim3 grid(blas_grid(c, nvec), c->nrhs_cur);
    const unsigned chunk = tile_chunk(c, prec);
    DWF_BLAS_DISPATCH(prec,
                      (xpay_kernel<float><<<grid, 256, 0, c->stream>>>((float4*)p, (const float4*)r, nvec, chunk, c->scalars,
                                                                     slot_cn, slot_c)),
                      (xpay_kernel<double><<<grid, 256, 0, c->stream>>>((double2*)p, (const double2*)r, nvec, chunk, c->scalars,
                                                                      slot_cn, slot_c)));
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

// elementwise kernels: nreal reals per system, all c->nrhs_cur systems of a batched field at once
dwf_status launch_axpy(dwf_ctx* c, void* y, const void* x, double a, int prec, size_t nreal) {
    const size_t nvec = nreal / (prec == DWF_F64 ? 2 : 4) * c->nrhs_cur;
    const int grid = blas_grid(c, nvec);
    DWF_BLAS_DISPATCH(prec, (axpy_kernel<float><<<grid, 256, 0, c->stream>>>((float4*)y, (const float4*)x, (float)a, nvec)),
                      (axpy_kernel<double><<<grid, 256, 0, c->stream>>>((double2*)y, (const double2*)x, a, nvec)));
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

dwf_status launch_sub(dwf_ctx* c, void* out, const void* a, const void* b, int prec, size_t nreal) {
    const size_t nvec = nreal / (prec == DWF_F64 ? 2 : 4) * c->nrhs_cur;
    const int grid = blas_grid(c, nvec);
    DWF_BLAS_DISPATCH(prec,
                      (sub_kernel<float><<<grid, 256, 0, c->stream>>>((float4*)out, (const float4*)a, (const float4*)b, nvec)),
                      (sub_kernel<double><<<grid, 256, 0, c->stream>>>((double2*)out, (const double2*)a, (const double2*)b, nvec)));
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

// r -= alpha (z + s0 p0), |r|^2 -> scalars[slot] with the stopping test of iteration `iter`   (fp64 fields)
dwf_status launch_ms_r(dwf_ctx* c, void* r, const void* z, const void* p0, size_t nreal, int slot_d, int slot, int iter) {
    const size_t nvec = nreal / 2;
    const int grid = blas_grid(c, nvec);
    dwf_status st = ensure_partials(c, grid);
    if (st != DWF_OK) return st;
    ms_alpha_kernel<<<1, 32, 0, c->stream>>>(c->ms_state, c->scalars, slot_d);
    ms_r_kernel<double><<<grid, 256, 0, c->stream>>>((double2*)r, (const double2*)z, (const double2*)p0, c->ms_state, nvec, c->partials);
    c->launches += 2;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return launch_reduce(c, grid, slot, iter);
}

// all shifts at once (fields i at x + i*nreal, p + i*nreal); |p_0|^2 -> state
dwf_status launch_ms_update(dwf_ctx* c, void* x, void* p, const void* r, size_t nreal, int slot_cn, int slot, int iter) {
    const size_t nvec = nreal / 2;
    const int grid = blas_grid(c, nvec);
    dwf_status st = ensure_partials(c, grid);
    if (st != DWF_OK) return st;
    ms_beta_kernel<<<1, 32, 0, c->stream>>>(c->ms_state, c->scalars, slot_cn);
    ms_update_kernel<double><<<grid, 256, 0, c->stream>>>((double2*)x, (double2*)p, (const double2*)r, nvec, c->ms_state, c->partials,
                                                          c->cg_conv, iter);
    c->launches += 2;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    st = launch_reduce(c, grid, slot, 0);
    if (st != DWF_OK) return st;
    ms_p0_kernel<<<1, 32, 0, c->stream>>>(c->ms_state, c->scalars, slot);
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

dwf_status launch_lincomb3(dwf_ctx* c, void* out, const void* x, const void* y, const void* z, double a, double b, double cc,
                           int prec, size_t nreal) {
    if (prec == DWF_F64) {
        const size_t nvec = nreal / 2;
        lincomb3_kernel<double><<<blas_grid(c, nvec), 256, 0, c->stream>>>((double2*)out, (const double2*)x, (const double2*)y,
                                                                        (const double2*)z, a, b, cc, nvec);
    } else {
        const size_t nvec = nreal / 4;
        lincomb3_kernel<float><<<blas_grid(c, nvec), 256, 0, c->stream>>>((float4*)out, (const float4*)x, (const float4*)y,
                                                                       (const float4*)z, (float)a, (float)b, (float)cc, nvec);
    }
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

}  // namespace dwf
