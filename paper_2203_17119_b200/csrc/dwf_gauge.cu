// Gauge preparation (step a0) and layout conversion kernels.
//
// Gauge prep implements PAPER.md:175 ("applies Dirichlet boundary conditions to its gauge field
// argument", reading C7): every link with x_mu mod B == B-1 is zeroed, then each OUTPUT site gets its 8
// leg matrices W_leg(x): forward U_mu(x), backward U_mu(x-mu)^dag, so that the hopping kernel reads all
// its links from its own lane (coalesced) and multiplies every leg the same way.  2-row compression
// (reading C10) keeps rows 0,1 of W; the antiperiodic sign is NOT baked in (it would be lost by the
// row-2 reconstruction) and is applied in the hopping kernel.
#include "dwf_layout.cuh"

namespace dwf {

template <typename R>
__global__ void gauge_prep_kernel(Geom g, const double* __restrict__ U, R* __restrict__ W, int parity, int ng,
                                  int kg_vw /* reals per link in the native array: KG*VW */, int vw, int cut0, int cut1,
                                  int cut2, int cut3) {
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;      // (native site, leg)
    if (gid >= g.Vh * 8) return;
    const int leg = gid & 7, site = gid >> 3;
    const int tile = site / g.TS, lane = site - tile * g.TS;
    const int mu = leg >> 1, dir = leg & 1;
    const int cut[4] = {cut0, cut1, cut2, cut3};
    Coord c = site_coords(g, tile, lane, parity);
    int y[4] = {c.x[0], c.x[1], c.x[2], c.x[3]};
    if (dir == 1) { y[mu] = c.x[mu] - 1; if (y[mu] < 0) y[mu] = g.L[mu] - 1; }
    const double* u = U + (lex_index(g, y) * 4 + mu) * 18;
    const bool zero = (cut[mu] > 0) && (y[mu] % cut[mu] == cut[mu] - 1);
    double w[18];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) {
            double re, im;
            if (dir == 0) { re = u[(r * 3 + cc) * 2]; im = u[(r * 3 + cc) * 2 + 1]; }
            else          { re = u[(cc * 3 + r) * 2]; im = -u[(cc * 3 + r) * 2 + 1]; }
            w[(r * 3 + cc) * 2] = zero ? 0.0 : re;
            w[(r * 3 + cc) * 2 + 1] = zero ? 0.0 : im;
        }
    // native: real index = (((tile*8 + leg)*KG + kg)*TS + lane)*VW + j, with i = kg*VW + j
    const int KG = kg_vw / vw;
    R* base = W + ((size_t)(tile * 8 + leg) * KG) * g.TS * vw;
    for (int i = 0; i < kg_vw; ++i) {
        const int kg = i / vw, j = i - kg * vw;
        base[((size_t)kg * g.TS + lane) * vw + j] = (i < ng) ? (R)w[i] : (R)0;
    }
}

// max over all links of |row2 - conj(row0 x row1)|_inf: what 2-row compression (reading C10) would get wrong.
// Non-negative doubles order like their bit patterns, so the maximum is an integer atomicMax.
__global__ void su3_defect_kernel(const double* __restrict__ U, long long nlinks, unsigned long long* __restrict__ worst) {
    double d = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nlinks; i += (long long)gridDim.x * blockDim.x) {
        const double* u = U + i * 18;
        for (int cidx = 0; cidx < 3; ++cidx) {
            const int a = (cidx + 1) % 3, b = (cidx + 2) % 3;
            const double re = (u[2 * a] * u[6 + 2 * b] - u[2 * a + 1] * u[6 + 2 * b + 1]) - (u[2 * b] * u[6 + 2 * a] - u[2 * b + 1] * u[6 + 2 * a + 1]);
            const double im = (u[2 * a] * u[6 + 2 * b + 1] + u[2 * a + 1] * u[6 + 2 * b]) - (u[2 * b] * u[6 + 2 * a + 1] + u[2 * b + 1] * u[6 + 2 * a]);
            d = fmax(d, fmax(fabs(u[12 + 2 * cidx] - re), fabs(u[12 + 2 * cidx + 1] + im)));
        }
    }
    if (!(d == d)) d = 1e300;      // NaN links
    atomicMax(worst, (unsigned long long)__double_as_longlong(d));
}

// 2-row storage is exact only for SU(3) links: refuse anything else instead of silently computing another operator
dwf_status check_su3(dwf_ctx* c, const double* Ucanon) {
    unsigned long long* w = reinterpret_cast<unsigned long long*>(c->scalars + (size_t)SLOT_T1 * MAXR);
    DWF_CUDA_CHECK(c, cudaMemsetAsync(w, 0, sizeof(*w), c->stream));
    const long long nlinks = 2LL * c->g.Vh * 4;
    su3_defect_kernel<<<c->num_sms * 4, 256, 0, c->stream>>>(Ucanon, nlinks, w);
    c->launches++;
    double d = 0.0;
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(&d, w, sizeof(d), cudaMemcpyDeviceToHost, c->stream));
    DWF_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (d > 1e-10) {
        char buf[200];
        snprintf(buf, sizeof(buf), "set_gauge: links are not SU(3) (max |row2 - conj(row0 x row1)| = %.3e): 2-row compression "
                                   "would change the operator; set option compress12 = 0", d);
        c->err = buf;
        return DWF_EINVAL;
    }
    return DWF_OK;
}

dwf_status launch_gauge_prep(dwf_ctx* c, const double* Ucanon) {
    const Geom& g = c->g;
    const int ng = c->compress12 ? 12 : 18;
    if (c->compress12) {
        dwf_status st = check_su3(c, Ucanon);
        if (st != DWF_OK) return st;
    }
    const int block = 128, grid = (g.Vh * 8 + block - 1) / block;
    const bool any_cut = c->cut[0] || c->cut[1] || c->cut[2] || c->cut[3];
    for (int set = 0; set < (any_cut && c->W64u[0] ? 2 : 1); ++set) {      // 0: with the Dirichlet cut, 1: without
        const int c0 = set ? 0 : c->cut[0], c1 = set ? 0 : c->cut[1], c2 = set ? 0 : c->cut[2], c3 = set ? 0 : c->cut[3];
        for (int par = 0; par < 2; ++par) {
            const int kg64 = (ng + 1) / 2 * 2, kg32 = (ng + 3) / 4 * 4;
            gauge_prep_kernel<double><<<grid, block, 0, c->stream>>>(geom_prec(c, DWF_F64), Ucanon,
                                                                     (double*)(set ? c->W64u[par] : c->W64[par]), par, ng, kg64, 2, c0, c1, c2, c3);
            gauge_prep_kernel<float><<<grid, block, 0, c->stream>>>(geom_prec(c, DWF_F32), Ucanon,
                                                                    (float*)(set ? c->W32u[par] : c->W32[par]), par, ng, kg32, 4, c0, c1, c2, c3);
            c->launches += 2;
        }
    }
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

void select_links(dwf_ctx* c, bool uncut) {
    if (c->links_uncut == uncut || !c->W64u[0]) return;
    for (int p = 0; p < 2; ++p) {
        void* t = c->W64[p]; c->W64[p] = c->W64u[p]; c->W64u[p] = t;
        t = c->W32[p]; c->W32[p] = c->W32u[p]; c->W32u[p] = t;
    }
    c->links_uncut = uncut;
}

// ---- spinor layout conversion: canonical <-> native, native f32 <-> native f64 ------------------
// real r = (spin*3+colour)*2+reim of site (tile, lane), slice s
template <typename R>
__device__ __forceinline__ size_t native_real_index(const Geom& g, int tile, int lane, int s, int r) {
    constexpr int VW = (sizeof(R) == 8) ? 2 : 4;
    constexpr int K = 24 / VW;
    const int k = r / VW, j = r - k * VW;
    return ((((size_t)tile * g.Ls + s) * K + k) * g.TS + lane) * VW + j;
}

// one thread per (native site, s).  canonical half field: [cb = lex/2][s][24]; FULL: [lex][s][24]
template <typename R, bool UNPACK>
__global__ void pack_kernel(Geom g, R* __restrict__ native, R* __restrict__ canon, int parity, int full) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)g.Vh * g.Ls) return;
    const int s = (int)(gid % g.Ls);
    const int site = (int)(gid / g.Ls);
    const int tile = site / g.TS, lane = site - tile * g.TS;
    Coord c = site_coords(g, tile, lane, parity);
    const long long lex = lex_index(g, c.x);
    const long long csite = full ? lex : (lex >> 1);
    R* cp = canon + (csite * g.Ls + s) * 24;
#pragma unroll
    for (int r = 0; r < 24; ++r) {
        const size_t ni = native_real_index<R>(g, tile, lane, s, r);
        if (UNPACK) cp[r] = native[ni]; else native[ni] = cp[r];
    }
}

// ---- domain and boundary projectors (eqs. 1-2, 8 PAPER.md:42-50, 87-89) --------------
// Omega = sites whose block indices floor(x_mu / B_mu), summed over the cut directions, are even.  The boundary projector
// P_dbar acts on the sites of Omega that have a cut link ("mask and shift by one in each direction"): forward link cut
// (x_mu mod B = B-1): the Omegabar neighbour reads (1 + gamma_mu) psi(x); backward link cut (x_mu mod B = 0): it reads
// (1 - gamma_mu) psi(x).  Shamir, one cut face at the site: (1 +- gamma_mu)/2; otherwise (Moebius: A = b5 + c5 Q mixes s
// and chirality; several faces): the identity on that site -- the smallest coordinate projector containing the minimal
// one.  gamma matrices: chiral basis of reading C1.
__device__ __forceinline__ void half_one_pm_gamma(int mu, double sg, const double (&v)[24], double (&o)[24]) {
    // gamma_mu psi, spin index a = 0..3, complex (re, im) per colour: rows listed as (source spin, factor) with factor in {1,-1,i,-i}
    // gx: (3,i)(2,i)(1,-i)(0,-i)  gy: (3,-1)(2,1)(1,1)(0,-1)  gz: (2,i)(3,-i)(0,-i)(1,i)  gt: (2,1)(3,1)(0,1)(1,1)
    const int src[4][4] = {{3, 2, 1, 0}, {3, 2, 1, 0}, {2, 3, 0, 1}, {2, 3, 0, 1}};
    const int fre[4][4] = {{0, 0, 0, 0}, {-1, 1, 1, -1}, {0, 0, 0, 0}, {1, 1, 1, 1}};      // real part of the factor
    const int fim[4][4] = {{1, 1, -1, -1}, {0, 0, 0, 0}, {1, -1, -1, 1}, {0, 0, 0, 0}};    // imaginary part of the factor
    for (int a = 0; a < 4; ++a) {
        const int b = src[mu][a];
        const double fr = fre[mu][a], fi = fim[mu][a];
        for (int cc = 0; cc < 3; ++cc) {
            const double xr = v[(b * 3 + cc) * 2], xi = v[(b * 3 + cc) * 2 + 1];
            const double gr = fr * xr - fi * xi, gi = fr * xi + fi * xr;
            o[(a * 3 + cc) * 2] = 0.5 * (v[(a * 3 + cc) * 2] + sg * gr);
            o[(a * 3 + cc) * 2 + 1] = 0.5 * (v[(a * 3 + cc) * 2 + 1] + sg * gi);
        }
    }
}

template <typename R>
__global__ void domain_project_kernel(Geom g, R* __restrict__ out, const R* __restrict__ in, int parity, int which, int cut0,
                                      int cut1, int cut2, int cut3, int shamir) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)g.Vh * g.Ls) return;
    const int s = (int)(gid % g.Ls);
    const int site = (int)(gid / g.Ls);
    const int tile = site / g.TS, lane = site - tile * g.TS;
    const int cut[4] = {cut0, cut1, cut2, cut3};
    const Coord c = site_coords(g, tile, lane, parity);
    int blk = 0, nface = 0, fmu = 0;
    double fsg = 0.0;
    for (int mu = 0; mu < 4; ++mu) {
        const int B = cut[mu];
        if (B <= 0) continue;
        blk += c.x[mu] / B;
        const int r = c.x[mu] % B;
        if (r == B - 1) { ++nface; fmu = mu; fsg = 1.0; }
        if (r == 0) { ++nface; fmu = mu; fsg = -1.0; }
    }
    const bool omega = (blk & 1) == 0;
    double v[24], o[24];
    for (int r = 0; r < 24; ++r) v[r] = (double)in[native_real_index<R>(g, tile, lane, s, r)];
    bool keep;
    if (which == 0) keep = omega;
    else if (which == 1) keep = !omega;
    else keep = omega && nface > 0;
    if (keep && which == 2 && shamir && nface == 1) {
        half_one_pm_gamma(fmu, fsg, v, o);
    } else {
        for (int r = 0; r < 24; ++r) o[r] = keep ? v[r] : 0.0;
    }
    for (int r = 0; r < 24; ++r) out[native_real_index<R>(g, tile, lane, s, r)] = (R)o[r];
}

dwf_status launch_domain_project(dwf_ctx* c, void* out, const void* in, int parity, int which, int prec) {
    const Geom g = geom_prec(c, prec);
    const long long n = (long long)g.Vh * g.Ls;
    const int block = 128, grid = (int)((n + block - 1) / block);
    const int shamir = (c->c5 == 0.0) ? 1 : 0;
    if (prec == DWF_F64)
        domain_project_kernel<double><<<grid, block, 0, c->stream>>>(g, (double*)out, (const double*)in, parity, which, c->cut[0],
                                                                     c->cut[1], c->cut[2], c->cut[3], shamir);
    else
        domain_project_kernel<float><<<grid, block, 0, c->stream>>>(g, (float*)out, (const float*)in, parity, which, c->cut[0],
                                                                    c->cut[1], c->cut[2], c->cut[3], shamir);
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

dwf_status launch_pack(dwf_ctx* c, void* native, const void* canon, int prec, int parity, bool unpack) {
    const Geom g = geom_prec(c, prec);
    const long long n = (long long)g.Vh * g.Ls;
    const int block = 128;
    const int grid = (int)((n + block - 1) / block);
    const int p0 = (parity == DWF_FULL) ? 0 : parity, p1 = (parity == DWF_FULL) ? 1 : parity;
    for (int par = p0; par <= p1; ++par) {
        const size_t off = (parity == DWF_FULL && par == 1) ? half_bytes(g, prec) : 0;
        void* nat = (char*)native + off;
        const int full = (parity == DWF_FULL);
        if (prec == DWF_F64) {
            if (unpack) pack_kernel<double, true><<<grid, block, 0, c->stream>>>(g, (double*)nat, (double*)canon, par, full);
            else pack_kernel<double, false><<<grid, block, 0, c->stream>>>(g, (double*)nat, (double*)canon, par, full);
        } else {
            if (unpack) pack_kernel<float, true><<<grid, block, 0, c->stream>>>(g, (float*)nat, (float*)canon, par, full);
            else pack_kernel<float, false><<<grid, block, 0, c->stream>>>(g, (float*)nat, (float*)canon, par, full);
        }
        c->launches++;
    }
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

// native -> native with a precision change; ACCUM: dst += src (used for x64 += e32)
template <typename RD, typename RS, bool ACCUM>
__global__ void convert_kernel(Geom g, RD* __restrict__ dst, const RS* __restrict__ src, int swz_d, int swz_s) {
    // one thread per (tile, s, lane, group of 4 reals)
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long n = (long long)g.Vh * g.Ls * 6;
    if (gid >= n) return;
    const int lane = (int)(gid % g.TS);
    long long r = gid / g.TS;
    const int q = (int)(r % 6);
    r /= 6;
    const int s = (int)(r % g.Ls);
    const int tile = (int)(r / g.Ls);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        // `lane` is the plain-order lane; a field in the XOR-rotated order (4^4 tiles) holds that site at lane ^ (tz << 1)
        const int rot = ((lane >> 3) & 3) << 1;
        const size_t si = native_real_index<RS>(g, tile, swz_s ? (lane ^ rot) : lane, s, q * 4 + j);
        const size_t di = native_real_index<RD>(g, tile, swz_d ? (lane ^ rot) : lane, s, q * 4 + j);
        if (ACCUM) dst[di] += (RD)src[si]; else dst[di] = (RD)src[si];
    }
}

dwf_status launch_convert(dwf_ctx* c, void* dst, int dprec, const void* src, int sprec, size_t nhalf_fields) {
    Geom g = c->g;
    g.Ls *= c->nrhs_cur;       // batched field: one long fifth dimension (dwf_internal.h)
    const long long n = (long long)g.Vh * g.Ls * 6;
    const int block = 256;
    const int grid = (int)((n + block - 1) / block);
    for (size_t h = 0; h < nhalf_fields; ++h) {
        void* d = (char*)dst + h * half_bytes(g, dprec);
        const void* s = (const char*)src + h * half_bytes(g, sprec);
        if (dprec == DWF_F32 && sprec == DWF_F64)
            convert_kernel<float, double, false><<<grid, block, 0, c->stream>>>(g, (float*)d, (const double*)s, 0, c->swz64);
        else if (dprec == DWF_F64 && sprec == DWF_F32)
            convert_kernel<double, float, false><<<grid, block, 0, c->stream>>>(g, (double*)d, (const float*)s, c->swz64, 0);
        else if (dprec == DWF_F64)
            convert_kernel<double, double, false><<<grid, block, 0, c->stream>>>(g, (double*)d, (const double*)s, 0, 0);
        else
            convert_kernel<float, float, false><<<grid, block, 0, c->stream>>>(g, (float*)d, (const float*)s, 0, 0);
        c->launches++;
    }
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

dwf_status launch_add_f32_to_f64(dwf_ctx* c, void* x64, const void* e32, size_t) {
    Geom g = c->g;
    g.Ls *= c->nrhs_cur;
    const long long n = (long long)g.Vh * g.Ls * 6;
    const int block = 256;
    const int grid = (int)((n + block - 1) / block);
    convert_kernel<double, float, true><<<grid, block, 0, c->stream>>>(g, (double*)x64, (const float*)e32, c->swz64, 0);
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

}  // namespace dwf
