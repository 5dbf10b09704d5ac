// C-ABI entry points (include/dwf.h), operator compositions and the CG drivers.
//
// Compositions (reading C5/C6; Meooe = -1/2 Dhop A, Mpc = Moo - Moe Mee^-1 Meo on odd sites):
//   Mpc x     = Moo x - 1/4 Dhop_o [A Mee^-1] Dhop_e [A] x                 (5 kernels; 4 on the fused path, where the
//                                                                            second Dhop adds Moo x in its epilogue)
//   Mpc^dag x = Moo^dag x - 1/4 A^dag Dhop^dag_o [Mee^-dag A^dag] Dhop^dag_e x   (4 kernels)
// where [..] are single fused 5-D table kernels and the final kernel also adds the Moo term and,
// inside CG, accumulates |Mpc p|^2.
#include <chrono>
#include <cmath>
#include <cstring>

#include "dwf_internal.h"

using namespace dwf;

namespace {

const int NWS = 10;

// The solver workspace (NWS half fields per precision, both precisions, whatever the caller goes on to use) is allocated
// once, at dwf_set_gauge, so that the vectors of dwf_cg / dwf_solve are never allocated inside a solve ("ctx owns
// ... CG workspace").  What is still allocated on first use, inside the first call that needs it, and then kept: the
// reduction partials (ensure_partials: a few KB, grows only when a larger grid or batch first appears), the multishift
// state and its nshift direction fields (dwf_multishift_cg), the two FULL fields of dwf_boundary_op, the device staging
// buffers of the *_host calls, and the batched workspace (dwf_mrhs_reserve, or the first batched call with a larger nrhs:
// NWSM fields of nrhs systems in both precisions).  dwf_norm2_static (dwf_noalloc.cu) is the one call that allocates nothing.
dwf_status ws_alloc_all(dwf_ctx* c) {
    for (int prec = 0; prec < 2; ++prec) {
        void** arr = (prec == DWF_F64) ? c->ws64 : c->ws32;
        for (int i = 0; i < NWS; ++i)
            if (!arr[i] && cudaMalloc(&arr[i], half_bytes(c->g, prec)) != cudaSuccess) {
                c->err = "cudaMalloc(workspace) failed";
                cudaGetLastError();
                return DWF_ENOMEM;
            }
    }
    return DWF_OK;
}

const int NWSM = 8;       // the batched Mpc / CG paths use workspace fields 0..7 only (8, 9 belong to dwf_solve)

void wsm_free(dwf_ctx* c) {
    for (int i = 0; i < NWSM; ++i) {
        if (c->wsm64[i]) cudaFree(c->wsm64[i]);
        if (c->wsm32[i]) cudaFree(c->wsm32[i]);
        c->wsm64[i] = c->wsm32[i] = nullptr;
    }
    c->mrhs_cap = 0;
}

dwf_status wsm_reserve(dwf_ctx* c, int nrhs) {
    if (nrhs <= c->mrhs_cap) return DWF_OK;
    wsm_free(c);
    for (int prec = 0; prec < 2; ++prec) {
        void** arr = (prec == DWF_F64) ? c->wsm64 : c->wsm32;
        for (int i = 0; i < NWSM; ++i)
            if (cudaMalloc(&arr[i], half_bytes(c->g, prec) * nrhs) != cudaSuccess) {
                cudaGetLastError();
                wsm_free(c);
                c->err = "cudaMalloc(batched workspace) failed";
                return DWF_ENOMEM;
            }
    }
    c->mrhs_cap = nrhs;
    return DWF_OK;
}

dwf_status ws_get(dwf_ctx* c, int prec, int idx, void** out) {
    void** arr = (c->nrhs_cur > 1) ? ((prec == DWF_F64) ? c->wsm64 : c->wsm32) : ((prec == DWF_F64) ? c->ws64 : c->ws32);
    if (!arr[idx] || (c->nrhs_cur > 1 && c->nrhs_cur > c->mrhs_cap)) { c->err = "workspace not allocated (call dwf_set_gauge)"; return DWF_ESTATE; }
    *out = arr[idx];
    return DWF_OK;
}

#define DWF_TRY(expr)                       \
    do {                                    \
        dwf_status _s = (expr);             \
        if (_s != DWF_OK) return _s;        \
    } while (0)

dwf_status need_gauge(dwf_ctx* c) {
    if (!c) return DWF_EINVAL;
    if (!c->gauge_set) { c->err = "gauge field not set (call dwf_set_gauge)"; return DWF_ESTATE; }
    return DWF_OK;
}

// sizes of ONE system's half field, and of the field the call in progress works on (all c->nrhs_cur systems)
size_t half_reals(const dwf_ctx* c) { return (size_t)c->g.Vh * c->g.Ls * 24; }
size_t cur_bytes(const dwf_ctx* c, int prec) { return half_bytes(c->g, prec) * c->nrhs_cur; }

// scalars[slot][0 .. nrhs_cur) -> host (synchronises the stream)
dwf_status read_slots(dwf_ctx* c, int slot, double* v) {
    const size_t o = (size_t)slot * MAXR;
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(c->scalars_host + o, c->scalars + o, sizeof(double) * c->nrhs_cur, cudaMemcpyDeviceToHost, c->stream));
    DWF_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    for (int j = 0; j < c->nrhs_cur; ++j) v[j] = c->scalars_host[o + j];
    return DWF_OK;
}
dwf_status read_slot(dwf_ctx* c, int slot, double* v) {      // system 0 only
    const size_t o = (size_t)slot * MAXR;
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(c->scalars_host + o, c->scalars + o, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    DWF_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    *v = c->scalars_host[o];
    return DWF_OK;
}

// out = Mpc in (dagger: Mpc^dag in) on odd half fields; norm_slot >= 0 also reduces |out|^2
dwf_status mpc_apply(dwf_ctx* c, void* out, const void* in, int dagger, int prec, int norm_slot) {
    void *t1, *t2;
    DWF_TRY(ws_get(c, prec, 0, &t1));
    DWF_TRY(ws_get(c, prec, 1, &t2));
    if (!dagger && dhop_fused_available(c)) {
        // the last step, Moo in - 1/4 (..) with the optional |.|^2, rides on the second Dhop (4 kernels instead of 5)
        DWF_TRY(launch_op5(c, t1, in, OP_A, nullptr, -1, 0.0, prec, -1));
        DWF_TRY(launch_dhop(c, t2, t1, DWF_EVEN, 0, prec));
        DWF_TRY(launch_op5(c, t1, t2, OP_A_MEEINV, nullptr, -1, 0.0, prec, -1));
        return launch_dhop_fused(c, out, t1, DWF_ODD, prec, in, -0.25, norm_slot);
    }
    if (!dagger) {
        DWF_TRY(launch_op5(c, t1, in, OP_A, nullptr, -1, 0.0, prec, -1));
        DWF_TRY(launch_dhop(c, t2, t1, DWF_EVEN, 0, prec));
        DWF_TRY(launch_op5(c, t1, t2, OP_A_MEEINV, nullptr, -1, 0.0, prec, -1));
        DWF_TRY(launch_dhop(c, t2, t1, DWF_ODD, 0, prec));
        DWF_TRY(launch_op5(c, out, in, OP_MEE, t2, -1, -0.25, prec, norm_slot));
    } else {
        DWF_TRY(launch_dhop(c, t1, in, DWF_EVEN, 1, prec));
        DWF_TRY(launch_op5(c, t2, t1, OP_MEEINVDAG_ADAG, nullptr, -1, 0.0, prec, -1));
        DWF_TRY(launch_dhop(c, t1, t2, DWF_ODD, 1, prec));
        DWF_TRY(launch_op5(c, out, in, OP_MEEDAG, t1, OP_ADAG, -0.25, prec, norm_slot));
    }
    return DWF_OK;
}

dwf_status mdagm_apply(dwf_ctx* c, void* out, const void* in, int prec) {
    void* q;
    DWF_TRY(ws_get(c, prec, 4, &q));
    DWF_TRY(mpc_apply(c, q, in, 0, prec, -1));
    return mpc_apply(c, out, q, 1, prec, -1);
}

// out_p = Mpp in_p + Meooe in_(1-p) on FULL fields (even half first)
dwf_status m_apply(dwf_ctx* c, void* out, const void* in, int dagger, int prec) {
    void *t1, *t2;
    DWF_TRY(ws_get(c, prec, 0, &t1));
    DWF_TRY(ws_get(c, prec, 1, &t2));
    const size_t hb = half_bytes(c->g, prec);
    for (int p = 0; p < 2; ++p) {
        const void* in_p = (const char*)in + p * hb;
        const void* in_q = (const char*)in + (1 - p) * hb;
        void* out_p = (char*)out + p * hb;
        if (!dagger) {
            DWF_TRY(launch_op5(c, t1, in_q, OP_A, nullptr, -1, 0.0, prec, -1));
            DWF_TRY(launch_dhop(c, t2, t1, p, 0, prec));
            DWF_TRY(launch_op5(c, out_p, in_p, OP_MEE, t2, -1, -0.5, prec, -1));
        } else {
            DWF_TRY(launch_dhop(c, t1, in_q, p, 1, prec));
            DWF_TRY(launch_op5(c, out_p, in_p, OP_MEEDAG, t1, OP_ADAG, -0.5, prec, -1));
        }
    }
    return DWF_OK;
}

// ---- CG on A = Mpc^dag Mpc for the c->nrhs_cur systems of a (batched) field (readings C8, C9) ------------------------
// The stopping test lives on the device (reduce_partials_kernel: cg_conv[j] = first iteration with |r_j|^2 <= cg_target[j])
// and the host enqueues iteration k + 1 before it has read the residual of iteration k: the GPU never waits for the host.
// Iteration k + 1 of a system that stopped at k only touches work vectors (cg_xp and cg_update leave x alone; the fused
// path also freezes p and r and zeroes the system's Dhop chain, the unfused path simply lets the recurrence of r and p run
// on), so the solution is the iterate of iteration k exactly, and the iteration count reported is k -- as in the oracle's loop.
struct CgRun {
    int n;                       // systems
    double target[MAXR];         // tol^2 |b|^2 (or the inner target), per system
    double c[MAXR];              // in: |r|^2 on entry; out: |r|^2 at the system's last counted iteration
    int iters[MAXR];             // out: iterations counted for the system in this run
    int launched;                // out: iterations enqueued (>= max iters[]: at most one more)
};

dwf_status cg_upload_state(dwf_ctx* c, CgRun& run, int slot_c) {
    double* h = c->scalars_host;
    int* hconv = reinterpret_cast<int*>(c->cn_ring + (size_t)CG_RING * MAXR + MAXR);
    double* htgt = c->cn_ring + (size_t)CG_RING * MAXR;
    for (int j = 0; j < run.n; ++j) {
        h[(size_t)slot_c * MAXR + j] = run.c[j];
        htgt[j] = run.target[j];
        hconv[j] = (run.c[j] <= run.target[j]) ? 0 : -1;          // already there: frozen from the start
    }
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(c->scalars + (size_t)slot_c * MAXR, h + (size_t)slot_c * MAXR, sizeof(double) * run.n, cudaMemcpyHostToDevice, c->stream));
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(c->cg_target, htgt, sizeof(double) * run.n, cudaMemcpyHostToDevice, c->stream));
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(c->cg_conv, hconv, sizeof(int) * run.n, cudaMemcpyHostToDevice, c->stream));
    DWF_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));        // the pinned staging is reused by the next upload
    return DWF_OK;
}

// On entry r holds the residuals and run.c their |.|^2; at most max_iter iterations are counted for any system.
dwf_status cg_iterate(dwf_ctx* c, int prec, void* x, void* r, int max_iter, CgRun& run) {
    void *p, *q, *z, *t1 = nullptr, *t2 = nullptr;
    DWF_TRY(ws_get(c, prec, 3, &p));
    DWF_TRY(ws_get(c, prec, 4, &q));
    DWF_TRY(ws_get(c, prec, 5, &z));
    DWF_TRY(ws_get(c, prec, 0, &t1));
    DWF_TRY(ws_get(c, prec, 1, &t2));
    const size_t n = half_reals(c);
    const int N = run.n;
    int slot_c = SLOT_C, slot_cn = SLOT_CN;
    DWF_TRY(cg_upload_state(c, run, slot_c));
    int conv[MAXR];
    bool all = true;
    for (int j = 0; j < N; ++j) {
        conv[j] = (run.c[j] <= run.target[j]) ? 0 : -1;
        run.iters[j] = 0;
        all = all && conv[j] >= 0;
    }
    run.launched = 0;
    if (all || max_iter <= 0) return DWF_OK;
    const bool fused = dhop_fused_available(c);
    // 8 kernels per iteration moving 23 half fields when the fused kernels apply: the second Dhop
    // carries q = Mee p - 1/4 (..) and |q|^2; one column kernel forms z = Mpc^dag's last step in registers and does
    // r -= alpha z, |r|^2; one does x += alpha p, p = r + beta p and the next A p.  Same operation order as the
    // unfused loop (reading C8).
    if (fused) DWF_TRY(launch_cg_xp(c, x, p, r, t1, prec, slot_c, SLOT_D, slot_cn, 1, 0));          // p = r, t1 = A p
    else DWF_CUDA_CHECK(c, cudaMemcpyAsync(p, r, cur_bytes(c, prec), cudaMemcpyDeviceToDevice, c->stream));
    int k = 0, decided = 0, stop_at = -1;
    // reads |r|^2 of iteration `it` (waits for it) and applies the stopping test; returns true when every system has stopped
    auto decide = [&](int it, dwf_status* st) -> bool {
        *st = DWF_OK;
        if (cudaEventSynchronize(c->cg_ev[it % CG_RING]) != cudaSuccess) { c->err = "cudaEventSynchronize failed"; *st = DWF_ECUDA; return true; }
        const double* cn = c->cn_ring + (size_t)(it % CG_RING) * MAXR;
        bool done = true;
        for (int j = 0; j < N; ++j) {
            if (conv[j] >= 0) continue;
            if (!(cn[j] == cn[j])) { c->err = "CG: NaN residual"; run.c[j] = cn[j]; *st = DWF_ECUDA; return true; }
            run.c[j] = cn[j];
            run.iters[j] = it;
            if (cn[j] <= run.target[j]) conv[j] = it; else done = false;
        }
        decided = it;
        return done;
    };
    dwf_status st = DWF_OK;
    while (k < max_iter) {
        ++k;
        if (fused) {
            DWF_TRY(launch_dhop(c, t2, t1, DWF_EVEN, 0, prec));
            DWF_TRY(launch_op5(c, t1, t2, OP_A_MEEINV, nullptr, -1, 0.0, prec, -1));
            DWF_TRY(launch_dhop_fused(c, q, t1, DWF_ODD, prec, p, -0.25, SLOT_D));           // q = Mpc p, d = |q|^2
            DWF_TRY(launch_dhop(c, t1, q, DWF_EVEN, 1, prec));
            DWF_TRY(launch_op5(c, t2, t1, OP_MEEINVDAG_ADAG, nullptr, -1, 0.0, prec, -1));
            DWF_TRY(launch_dhop(c, t1, t2, DWF_ODD, 1, prec));
            DWF_TRY(launch_cg_r(c, r, q, t1, -0.25, prec, slot_c, SLOT_D, slot_cn, k));     // r -= a Mpc^dag q; stopping test
        } else {
            DWF_TRY(mpc_apply(c, q, p, 0, prec, SLOT_D));                 // q = Mpc p, d = |q|^2
            DWF_TRY(mpc_apply(c, z, q, 1, prec, -1));                     // z = Mpc^dag q
            DWF_TRY(launch_cg_update(c, x, r, p, z, prec, n, slot_c, SLOT_D, slot_cn, k));   // x += a p; r -= a z; test
        }
        DWF_CUDA_CHECK(c, cudaMemcpyAsync(c->cn_ring + (size_t)(k % CG_RING) * MAXR, c->scalars + (size_t)slot_cn * MAXR,
                                          sizeof(double) * N, cudaMemcpyDeviceToHost, c->stream));
        DWF_CUDA_CHECK(c, cudaEventRecord(c->cg_ev[k % CG_RING], c->stream));
        if (fused) DWF_TRY(launch_cg_xp(c, x, p, r, t1, prec, slot_c, SLOT_D, slot_cn, 0, k));      // x += a p; p = r + b p; t1 = A p
        else DWF_TRY(launch_xpay(c, p, r, prec, n, slot_cn, slot_c));                           // p = r + (cn/c) p
        { int t = slot_c; slot_c = slot_cn; slot_cn = t; }
        if (k >= 2 && decide(k - 1, &st)) { stop_at = k - 1; break; }
    }
    if (st != DWF_OK) return st;
    while (stop_at < 0 && decided < k) {
        if (decide(decided + 1, &st)) stop_at = decided;
        if (st != DWF_OK) return st;
    }
    run.launched = k;
    return DWF_OK;
}

// |v_j|^2 of every system of the field in progress
dwf_status norm2_host(dwf_ctx* c, const void* v, int prec, double* out) {
    DWF_TRY(launch_norm2(c, v, prec, half_reals(c), SLOT_T0));
    return read_slots(c, SLOT_T0, out);
}

// r = b - A x (fp64), returns |r_j|^2
dwf_status true_residual(dwf_ctx* c, void* r, const void* b, const void* x, double* rn2) {
    void* ax;
    DWF_TRY(ws_get(c, DWF_F64, 6, &ax));
    DWF_TRY(mdagm_apply(c, ax, x, DWF_F64));
    DWF_TRY(launch_sub(c, r, b, ax, DWF_F64, half_reals(c)));
    return norm2_host(c, r, DWF_F64, rn2);
}

// zero the systems of a batched fp64 field whose right-hand side vanishes (x_j = 0 is the solution)
dwf_status zero_systems(dwf_ctx* c, void* x, const double* bn2) {
    const size_t chunk = (size_t)c->g.Ls * 12 * c->g.TS * 16;       // bytes of one tile of one system
    for (int j = 0; j < c->nrhs_cur; ++j)
        if (bn2[j] == 0.0)
            DWF_CUDA_CHECK(c, cudaMemset2DAsync((char*)x + j * chunk, chunk * c->nrhs_cur, 0, chunk, c->g.ntiles, c->stream));
    return DWF_OK;
}

// info: one entry per system
dwf_status cg_f64(dwf_ctx* c, void* x, const void* b, double tol, int max_iter, int use_guess, dwf_cg_info* info) {
    void* r;
    DWF_TRY(ws_get(c, DWF_F64, 2, &r));
    const int N = c->nrhs_cur;
    const size_t hb = cur_bytes(c, DWF_F64);
    double bn2[MAXR];
    DWF_TRY(norm2_host(c, b, DWF_F64, bn2));
    if (!use_guess) DWF_CUDA_CHECK(c, cudaMemsetAsync(x, 0, hb, c->stream));
    else DWF_TRY(zero_systems(c, x, bn2));
    bool any = false;
    for (int j = 0; j < N; ++j) any = any || bn2[j] != 0.0;
    if (!any) return DWF_OK;
    CgRun run;
    run.n = N;
    for (int j = 0; j < N; ++j) run.target[j] = tol * tol * bn2[j];
    int iters[MAXR] = {}, restarts = 0, most = 0;       // most: the largest iteration count of any system so far
    double rt[MAXR];
    bool conv = false;
    for (;;) {
        if (use_guess || restarts > 0) {
            DWF_TRY(true_residual(c, r, b, x, run.c));
        } else {
            DWF_CUDA_CHECK(c, cudaMemcpyAsync(r, b, hb, cudaMemcpyDeviceToDevice, c->stream));
            for (int j = 0; j < N; ++j) run.c[j] = bn2[j];
        }
        // the budget is spent by COUNTED iterations (as in the oracle's loop), not by enqueued ones: the iteration the host
        // runs ahead of the stopping test costs nothing
        DWF_TRY(cg_iterate(c, DWF_F64, x, r, max_iter - most, run));
        for (int j = 0; j < N; ++j) {
            iters[j] += run.iters[j];
            most = iters[j] > most ? iters[j] : most;
            info[j].resid_iter = bn2[j] > 0 ? std::sqrt(run.c[j] / bn2[j]) : 0.0;
        }
        void* tr;
        DWF_TRY(ws_get(c, DWF_F64, 7, &tr));
        double tn2[MAXR];
        DWF_TRY(true_residual(c, tr, b, x, tn2));
        conv = true;
        for (int j = 0; j < N; ++j) {
            rt[j] = bn2[j] > 0 ? std::sqrt(tn2[j] / bn2[j]) : 0.0;
            conv = conv && rt[j] <= tol;
        }
        if (conv || most >= max_iter) break;
        ++restarts;
    }
    for (int j = 0; j < N; ++j) {
        info[j].iters_total = iters[j];
        info[j].restarts = restarts;
        info[j].resid_true = rt[j];
    }
    return conv ? DWF_OK : DWF_ENOTCONV;
}

// reading C9: fp64 outer defect correction around an fp32 inner CG
dwf_status cg_mixed(dwf_ctx* c, void* x, const void* b, double tol, int max_iter, int use_guess, dwf_cg_info* info) {
    void *r, *r32, *e32;
    DWF_TRY(ws_get(c, DWF_F64, 2, &r));
    DWF_TRY(ws_get(c, DWF_F32, 2, &r32));
    DWF_TRY(ws_get(c, DWF_F32, 6, &e32));
    const int N = c->nrhs_cur;
    const size_t hb = cur_bytes(c, DWF_F64), hb32 = cur_bytes(c, DWF_F32);
    double bn2[MAXR];
    DWF_TRY(norm2_host(c, b, DWF_F64, bn2));
    if (!use_guess) DWF_CUDA_CHECK(c, cudaMemsetAsync(x, 0, hb, c->stream));
    else DWF_TRY(zero_systems(c, x, bn2));
    bool any = false;
    for (int j = 0; j < N; ++j) any = any || bn2[j] != 0.0;
    if (!any) return DWF_OK;
    int iters[MAXR] = {}, restarts = 0, most = 0, outer[MAXR] = {};      // most: as in cg_f64, counted iterations
    double rt[MAXR];
    bool conv = false;
    for (;;) {
        double rn2[MAXR];
        DWF_TRY(true_residual(c, r, b, x, rn2));
        conv = true;
        for (int j = 0; j < N; ++j) {
            rt[j] = bn2[j] > 0 ? std::sqrt(rn2[j] / bn2[j]) : 0.0;
            conv = conv && rt[j] <= tol;
        }
        if (conv || restarts >= c->max_restarts || most >= max_iter) break;
        DWF_TRY(launch_convert(c, r32, DWF_F32, r, DWF_F64, 1));
        CgRun run;
        run.n = N;
        DWF_TRY(norm2_host(c, r32, DWF_F32, run.c));
        DWF_CUDA_CHECK(c, cudaMemsetAsync(e32, 0, hb32, c->stream));
        double r32n2[MAXR];
        for (int j = 0; j < N; ++j) {
            r32n2[j] = run.c[j];
            if (rt[j] <= tol) { run.target[j] = 1e300; continue; }       // this system is done: frozen, e_j stays 0
            const double delta = std::fmax(c->inner_tol, tol * std::sqrt(bn2[j] / rn2[j]));
            run.target[j] = delta * delta * r32n2[j];
            ++outer[j];
        }
        DWF_TRY(cg_iterate(c, DWF_F32, e32, r32, max_iter - most, run));
        for (int j = 0; j < N; ++j) {
            iters[j] += run.iters[j];
            most = iters[j] > most ? iters[j] : most;
            if (r32n2[j] > 0 && rt[j] > tol) info[j].resid_iter = std::sqrt(run.c[j] / r32n2[j]);
        }
        DWF_TRY(launch_add_f32_to_f64(c, x, e32, 0));
        ++restarts;
    }
    for (int j = 0; j < N; ++j) {
        info[j].iters_total = iters[j];
        info[j].iters_inner = iters[j];
        info[j].restarts = outer[j];
        info[j].resid_true = rt[j];
    }
    return conv ? DWF_OK : DWF_ENOTCONV;
}

double now_s() {
    return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

dwf_status stage_get(dwf_ctx* c, int idx, size_t bytes, void** out) {
    if (c->stage_bytes[idx] < bytes) {
        if (c->stage_dev[idx]) cudaFree(c->stage_dev[idx]);
        c->stage_dev[idx] = nullptr;
        c->stage_bytes[idx] = 0;
        if (cudaMalloc(&c->stage_dev[idx], bytes) != cudaSuccess) { c->err = "cudaMalloc(stage) failed"; cudaGetLastError(); return DWF_ENOMEM; }
        c->stage_bytes[idx] = bytes;
    }
    *out = c->stage_dev[idx];
    return DWF_OK;
}

void choose_tiles(dwf_ctx* c) {
    Geom& g = c->g;
    for (int mu = 0; mu < 4; ++mu) {
        int t = c->tile_opt[mu];
        if (t <= 0) t = (g.L[mu] % 4 == 0) ? 4 : 2;
        g.T[mu] = t;
        g.NT[mu] = g.L[mu] / t;
    }
    g.swz = 0;
    c->swz64 = (g.T[0] == 4 && g.T[1] == 4 && g.T[2] == 4 && g.T[3] == 4) ? 1 : 0;
    g.TS = g.T[0] * g.T[1] * g.T[2] * g.T[3] / 2;
    g.ntiles = g.NT[0] * g.NT[1] * g.NT[2] * g.NT[3];
    g.Vh = g.ntiles * g.TS;
}

}  // namespace

extern "C" {

const char* dwf_version(void) { return "dwf_b200 0.1 (sm_100a)"; }

dwf_status dwf_create(dwf_ctx** out, const int dims[4], int Ls, double M5, double mf, double b5, double c5,
                      const int dirichlet_cut[4]) {
    if (!out || !dims) return DWF_EINVAL;
    *out = nullptr;
    if (Ls < 1 || Ls > 32) return DWF_EINVAL;
    long long V = 1;
    for (int mu = 0; mu < 4; ++mu) {
        if (dims[mu] < 2 || (dims[mu] & 1)) return DWF_EINVAL;
        if (dirichlet_cut) {
            int B = dirichlet_cut[mu];
            if (B < 0 || (B > 0 && dims[mu] % B != 0)) return DWF_EINVAL;
        }
        V *= dims[mu];
    }
    if (V / 2 * Ls * 12 >= (1LL << 31)) return DWF_EINVAL;   // 32-bit vector indices inside the kernels
    const double bee = 1.0 + b5 * (4.0 - M5);
    if (bee == 0.0) return DWF_EINVAL;
    dwf_ctx* c = new (std::nothrow) dwf_ctx();
    if (!c) return DWF_ENOMEM;
    for (int mu = 0; mu < 4; ++mu) {
        c->g.L[mu] = dims[mu];
        c->cut[mu] = dirichlet_cut ? dirichlet_cut[mu] : 0;
    }
    c->g.Ls = Ls;
    c->g.antiperiodic_t = 1;
    cudaGetDevice(&c->device);
    if (cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess || c->num_sms < 1) {
        cudaGetLastError();
        c->num_sms = 148;
    }
    c->M5 = M5; c->mf = mf; c->b5 = b5; c->c5 = c5;
    choose_tiles(c);
    build_tables(c);
    bool ok = cudaMalloc(&c->scalars, sizeof(double) * NSLOTS * MAXR) == cudaSuccess &&
              cudaMallocHost(&c->scalars_host, sizeof(double) * NSLOTS * MAXR) == cudaSuccess &&
              cudaMalloc(&c->cg_target, sizeof(double) * MAXR) == cudaSuccess &&
              cudaMalloc(&c->cg_conv, sizeof(int) * MAXR) == cudaSuccess &&
              // |r|^2 ring of the last CG_RING iterations, then the staging of cg_target and cg_conv
              cudaMallocHost(&c->cn_ring, sizeof(double) * (CG_RING + 2) * MAXR) == cudaSuccess &&
              cudaMemset(c->scalars, 0, sizeof(double) * NSLOTS * MAXR) == cudaSuccess &&
              cudaMemset(c->cg_conv, 0xff, sizeof(int) * MAXR) == cudaSuccess;
    for (int i = 0; i < CG_RING && ok; ++i) ok = cudaEventCreateWithFlags(&c->cg_ev[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        dwf_destroy(c);
        return DWF_ECUDA;
    }
    // device tables [op][chirality][Ls*Ls]
    const size_t nt = (size_t)OP5_COUNT * 2 * Ls * Ls;
    std::vector<double> h64(nt);
    std::vector<float> h32(nt);
    for (int op = 0; op < OP5_COUNT; ++op)
        for (int ch = 0; ch < 2; ++ch)
            for (int s = 0; s < Ls; ++s)
                for (int t = 0; t < Ls; ++t) {
                    const double v = (ch == 0 ? c->tab[op].p : c->tab[op].m)[s * 32 + t];
                    const size_t i = (((size_t)op * 2 + ch) * Ls + s) * Ls + t;
                    h64[i] = v;
                    h32[i] = (float)v;
                }
    if (cudaMalloc(&c->dtab.d64, nt * sizeof(double)) != cudaSuccess || cudaMalloc(&c->dtab.d32, nt * sizeof(float)) != cudaSuccess) {
        cudaGetLastError();
        dwf_destroy(c);
        return DWF_ENOMEM;
    }
    if (cudaMemcpy(c->dtab.d64, h64.data(), nt * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(c->dtab.d32, h32.data(), nt * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        dwf_destroy(c);
        return DWF_ECUDA;
    }
    *out = c;
    return DWF_OK;
}

dwf_status dwf_destroy(dwf_ctx* c) {
    DeviceGuard _dev(c);
    if (!c) return DWF_EINVAL;
    for (int p = 0; p < 2; ++p) {
        if (c->W64[p]) cudaFree(c->W64[p]);
        if (c->W32[p]) cudaFree(c->W32[p]);
        if (c->stage_dev[p]) cudaFree(c->stage_dev[p]);
        if (c->W64u[p]) cudaFree(c->W64u[p]);
        if (c->W32u[p]) cudaFree(c->W32u[p]);
    }
    if (c->bnd_ws) cudaFree(c->bnd_ws);
    for (int i = 0; i < NWS; ++i) {
        if (c->ws64[i]) cudaFree(c->ws64[i]);
        if (c->ws32[i]) cudaFree(c->ws32[i]);
    }
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    pipe_tables_free(c);
    tma_state_free(c);
    if (c->ms_p) cudaFree(c->ms_p);
    if (c->ms_state) cudaFree(c->ms_state);
    if (c->partials) cudaFree(c->partials);
    if (c->scalars) cudaFree(c->scalars);
    if (c->scalars_host) cudaFreeHost(c->scalars_host);
    if (c->cg_target) cudaFree(c->cg_target);
    if (c->cg_conv) cudaFree(c->cg_conv);
    if (c->cn_ring) cudaFreeHost(c->cn_ring);
    for (int i = 0; i < CG_RING; ++i)
        if (c->cg_ev[i]) cudaEventDestroy(c->cg_ev[i]);
    wsm_free(c);
    if (c->dtab.d64) cudaFree(c->dtab.d64);
    if (c->dtab.d32) cudaFree(c->dtab.d32);
    cudaGetLastError();
    delete c;
    return DWF_OK;
}

dwf_status dwf_set_option(dwf_ctx* c, const char* key, double val) {
    DeviceGuard _dev(c);
    if (!c || !key) return DWF_EINVAL;
    const std::string k(key);
    const bool pre_gauge = (k == "antiperiodic_t" || k == "compress12" || k.rfind("tile_", 0) == 0);
    if (pre_gauge && c->gauge_set) { c->err = "option '" + k + "' must be set before dwf_set_gauge"; return DWF_ESTATE; }
    if (k == "antiperiodic_t") c->g.antiperiodic_t = (val != 0.0);
    else if (k == "compress12") c->compress12 = (val != 0.0);
    else if (k == "tile_x" || k == "tile_y" || k == "tile_z" || k == "tile_t") {
        const int mu = (k == "tile_x") ? 0 : (k == "tile_y") ? 1 : (k == "tile_z") ? 2 : 3;
        const int t = (int)val;
        if (t < 1 || c->g.L[mu] % t != 0 || (mu == 0 && (t & 1))) { c->err = "bad tile extent"; return DWF_EINVAL; }
        const int old = c->tile_opt[mu];
        c->tile_opt[mu] = t;
        choose_tiles(c);
        if (c->g.TS > 1024) { c->tile_opt[mu] = old; choose_tiles(c); c->err = "tile too large"; return DWF_EINVAL; }
    } else if (k == "inner_tol") c->inner_tol = val;
    else if (k == "max_restarts") c->max_restarts = (int)val;
    else if (k == "dhop_kernel") c->dhop_kernel = (int)val;
    else if (k == "fuse") c->fuse = (val != 0.0);
    else if (k == "dhop_dynamic") { if (val < 0 || val > 1) return DWF_EINVAL; c->dhop_dynamic = (int)val; }
    else if (k == "time_dhop") {       // (re)start per-launch event timing of the Dhop kernel
        DWF_TRY(dhop_timing_flush(c));
        c->time_dhop = (val != 0.0);
        c->dhop_ms = 0.0;
        c->dhop_bytes = 0.0;
        c->dhop_timed = 0;
    }
    else { c->err = "unknown option '" + k + "'"; return DWF_EINVAL; }
    return DWF_OK;
}

dwf_status dwf_get_option(const dwf_ctx* c, const char* key, double* val) {
    DeviceGuard _dev(c);
    if (!c || !key || !val) return DWF_EINVAL;
    const std::string k(key);
    if (k == "dhop_ms" || k == "dhop_timed" || k == "dhop_bytes") {   // synchronises: folds the pending event pairs
        dwf_ctx* m = const_cast<dwf_ctx*>(c);
        DWF_TRY(dhop_timing_flush(m));
        *val = (k == "dhop_ms") ? m->dhop_ms : (k == "dhop_bytes" ? m->dhop_bytes : (double)m->dhop_timed);
        return DWF_OK;
    }
    if (k == "antiperiodic_t") *val = c->g.antiperiodic_t;
    else if (k == "compress12") *val = c->compress12;
    else if (k == "tile_x") *val = c->g.T[0];
    else if (k == "tile_y") *val = c->g.T[1];
    else if (k == "tile_z") *val = c->g.T[2];
    else if (k == "tile_t") *val = c->g.T[3];
    else if (k == "inner_tol") *val = c->inner_tol;
    else if (k == "max_restarts") *val = c->max_restarts;
    else if (k == "time_dhop") *val = c->time_dhop;
    else if (k == "dhop_kernel") *val = c->dhop_kernel;
    else if (k == "dhop_dynamic") *val = c->dhop_dynamic;
    else if (k == "fuse") *val = c->fuse;
    else if (k == "fused_active") *val = dhop_fused_available(c) ? 1.0 : 0.0;
    else if (k == "mrhs_reserved") *val = c->mrhs_cap;
    else return DWF_EINVAL;
    return DWF_OK;
}

dwf_status dwf_set_stream(dwf_ctx* c, void* s) {
    DeviceGuard _dev(c);
    if (!c) return DWF_EINVAL;
    c->stream = (cudaStream_t)s;
    return DWF_OK;
}

dwf_status dwf_set_gauge(dwf_ctx* c, const void* U) {
    DeviceGuard _dev(c);
    if (!c || !U) return DWF_EINVAL;
    const Geom& g = c->g;
    const int ng = c->compress12 ? 12 : 18;
    const size_t b64 = (size_t)g.Vh * 8 * ((ng + 1) / 2) * 16, b32 = (size_t)g.Vh * 8 * ((ng + 3) / 4) * 16;
    for (int p = 0; p < 2; ++p) {
        if (c->W64[p] && c->wbytes64 != b64) { cudaFree(c->W64[p]); c->W64[p] = nullptr; }
        if (c->W32[p] && c->wbytes32 != b32) { cudaFree(c->W32[p]); c->W32[p] = nullptr; }
        if (!c->W64[p] && cudaMalloc(&c->W64[p], b64) != cudaSuccess) { cudaGetLastError(); c->err = "cudaMalloc(gauge) failed"; return DWF_ENOMEM; }
        if (!c->W32[p] && cudaMalloc(&c->W32[p], b32) != cudaSuccess) { cudaGetLastError(); c->err = "cudaMalloc(gauge) failed"; return DWF_ENOMEM; }
    }
    const bool any_cut = c->cut[0] || c->cut[1] || c->cut[2] || c->cut[3];
    select_links(c, false);
    for (int p = 0; p < 2 && any_cut; ++p) {      // the same field without the cut, for the boundary operators (eqs. 8-14)
        if (c->W64u[p] && c->wbytes64 != b64) { cudaFree(c->W64u[p]); c->W64u[p] = nullptr; }
        if (c->W32u[p] && c->wbytes32 != b32) { cudaFree(c->W32u[p]); c->W32u[p] = nullptr; }
        if (!c->W64u[p] && cudaMalloc(&c->W64u[p], b64) != cudaSuccess) { cudaGetLastError(); c->err = "cudaMalloc(gauge) failed"; return DWF_ENOMEM; }
        if (!c->W32u[p] && cudaMalloc(&c->W32u[p], b32) != cudaSuccess) { cudaGetLastError(); c->err = "cudaMalloc(gauge) failed"; return DWF_ENOMEM; }
    }
    c->wbytes64 = b64;
    c->wbytes32 = b32;
    DWF_TRY(ws_alloc_all(c));
    DWF_TRY(launch_gauge_prep(c, (const double*)U));
    DWF_TRY(pipe_tables_upload(c));
    DWF_TRY(tma_state_build(c));
    c->gauge_set = true;
    return DWF_OK;
}

size_t dwf_field_bytes(const dwf_ctx* c, dwf_prec prec, dwf_parity parity) {
    DeviceGuard _dev(c);
    if (!c) return 0;
    return half_bytes(c->g, prec) * (parity == DWF_FULL ? 2 : 1);
}

dwf_status dwf_pack(dwf_ctx* c, void* native, const void* canon, dwf_prec prec, dwf_parity parity) {
    DeviceGuard _dev(c);
    if (!c || !native || !canon) return DWF_EINVAL;
    return launch_pack(c, native, canon, prec, parity, false);
}
dwf_status dwf_unpack(dwf_ctx* c, void* canon, const void* native, dwf_prec prec, dwf_parity parity) {
    DeviceGuard _dev(c);
    if (!c || !native || !canon) return DWF_EINVAL;
    return launch_pack(c, const_cast<void*>(native), canon, prec, parity, true);
}
dwf_status dwf_convert(dwf_ctx* c, void* dst, dwf_prec dp, const void* src, dwf_prec sp, dwf_parity parity) {
    DeviceGuard _dev(c);
    if (!c || !dst || !src || dst == src) return DWF_EINVAL;
    return launch_convert(c, dst, dp, src, sp, parity == DWF_FULL ? 2 : 1);
}

dwf_status dwf_dhop(dwf_ctx* c, void* out, const void* in, dwf_parity out_parity, int dagger, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out || !in || out == in) { c->err = "dhop: null or aliased pointers"; return DWF_EINVAL; }
    if (out_parity == DWF_FULL) {
        const size_t hb = half_bytes(c->g, prec);
        DWF_TRY(launch_dhop(c, out, (const char*)in + hb, DWF_EVEN, dagger, prec));
        return launch_dhop(c, (char*)out + hb, in, DWF_ODD, dagger, prec);
    }
    return launch_dhop(c, out, in, out_parity, dagger, prec);
}

static dwf_status op5_public(dwf_ctx* c, void* out, const void* in, dwf_parity parity, int op, dwf_prec prec) {
    if (!c || !out || !in) return DWF_EINVAL;
    if (out == in) { c->err = "5-D operator: out must not alias in"; return DWF_EINVAL; }
    const int nh = (parity == DWF_FULL) ? 2 : 1;
    const size_t hb = half_bytes(c->g, prec);
    for (int h = 0; h < nh; ++h) DWF_TRY(launch_op5(c, (char*)out + h * hb, (const char*)in + h * hb, op, nullptr, -1, 0.0, prec, -1));
    return DWF_OK;
}
dwf_status dwf_meooe5d(dwf_ctx* c, void* out, const void* in, dwf_parity par, int dagger, dwf_prec prec) {
    DeviceGuard _dev(c);
    return op5_public(c, out, in, par, dagger ? OP_ADAG : OP_A, prec);
}
dwf_status dwf_mooee(dwf_ctx* c, void* out, const void* in, dwf_parity par, int dagger, dwf_prec prec) {
    DeviceGuard _dev(c);
    return op5_public(c, out, in, par, dagger ? OP_MEEDAG : OP_MEE, prec);
}
dwf_status dwf_mooee_inv(dwf_ctx* c, void* out, const void* in, dwf_parity par, int dagger, dwf_prec prec) {
    DeviceGuard _dev(c);
    return op5_public(c, out, in, par, dagger ? OP_MEEINVDAG : OP_MEEINV, prec);
}

dwf_status dwf_m(dwf_ctx* c, void* out, const void* in, int dagger, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out || !in || out == in) { c->err = "m: null or aliased pointers"; return DWF_EINVAL; }
    return m_apply(c, out, in, dagger, prec);
}
dwf_status dwf_mpc(dwf_ctx* c, void* out, const void* in, int dagger, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out || !in || out == in) { c->err = "mpc: null or aliased pointers"; return DWF_EINVAL; }
    return mpc_apply(c, out, in, dagger, prec, -1);
}
dwf_status dwf_mdagm(dwf_ctx* c, void* out, const void* in, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out || !in || out == in) { c->err = "mdagm: null or aliased pointers"; return DWF_EINVAL; }
    return mdagm_apply(c, out, in, prec);
}

dwf_status dwf_norm2(dwf_ctx* c, const void* v, dwf_prec prec, dwf_parity parity, double* result) {
    DeviceGuard _dev(c);
    if (!c || !v || !result) return DWF_EINVAL;
    const size_t n = half_reals(c) * (parity == DWF_FULL ? 2 : 1);
    DWF_TRY(launch_norm2(c, v, prec, n, SLOT_T0));
    return read_slot(c, SLOT_T0, result);
}

dwf_status dwf_cg(dwf_ctx* c, void* x, const void* b, double tol, int max_iter, dwf_cg_mode mode, int use_guess,
                  dwf_cg_info* info) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    dwf_cg_info local;
    if (!info) info = &local;
    memset(info, 0, sizeof(*info));
    if (!x || !b || x == b || tol <= 0.0 || max_iter < 0) { c->err = "cg: bad arguments"; return DWF_EINVAL; }
    const long long l0 = c->launches;
    const double t0 = now_s();
    dwf_status st = (mode == DWF_CG_MIXED) ? cg_mixed(c, x, b, tol, max_iter, use_guess, info)
                                           : cg_f64(c, x, b, tol, max_iter, use_guess, info);
    cudaStreamSynchronize(c->stream);
    info->seconds = now_s() - t0;
    info->launches = (int)(c->launches - l0);
    if (st == DWF_ENOTCONV) c->err = "cg: max_iter reached";
    return st;
}

// ---- batched (multi right-hand side) fields and operators --------------------------------------
namespace {
struct BatchGuard {       // the batch count is only ever visible inside one ABI call
    dwf_ctx* c;
    BatchGuard(dwf_ctx* cc, int n) : c(cc) { c->nrhs_cur = n; }
    ~BatchGuard() { c->nrhs_cur = 1; }
};
dwf_status mrhs_ok(dwf_ctx* c, int nrhs) {
    if (nrhs < 1 || nrhs > MAXR) { c->err = "mrhs: nrhs must be 1..16"; return DWF_EINVAL; }
    if ((long long)c->g.Vh * c->g.Ls * 12 * nrhs >= (1LL << 31)) { c->err = "mrhs: batched field too large for 32-bit vector indices"; return DWF_EINVAL; }
    return DWF_OK;
}
}  // namespace

dwf_status dwf_mrhs_reserve(dwf_ctx* c, int nrhs) {
    DeviceGuard _dev(c);
    if (!c) return DWF_EINVAL;
    DWF_TRY(mrhs_ok(c, nrhs));
    return nrhs > 1 ? wsm_reserve(c, nrhs) : DWF_OK;
}

size_t dwf_mrhs_field_bytes(const dwf_ctx* c, int nrhs, dwf_prec prec) {
    if (!c || nrhs < 1) return 0;
    return half_bytes(c->g, prec) * nrhs;
}

// strided copies between system j of a batched half field and a single native half field (tile by tile)
dwf_status dwf_mrhs_insert(dwf_ctx* c, void* batched, int nrhs, int j, const void* single, dwf_prec prec) {
    DeviceGuard _dev(c);
    if (!c || !batched || !single) return DWF_EINVAL;
    DWF_TRY(mrhs_ok(c, nrhs));
    if (j < 0 || j >= nrhs) { c->err = "mrhs: system index out of range"; return DWF_EINVAL; }
    const size_t chunk = half_bytes(c->g, prec) / c->g.ntiles;        // bytes of one tile of one system
    DWF_CUDA_CHECK(c, cudaMemcpy2DAsync((char*)batched + j * chunk, chunk * nrhs, single, chunk, chunk, c->g.ntiles,
                                        cudaMemcpyDeviceToDevice, c->stream));
    return DWF_OK;
}
dwf_status dwf_mrhs_extract(dwf_ctx* c, void* single, const void* batched, int nrhs, int j, dwf_prec prec) {
    DeviceGuard _dev(c);
    if (!c || !batched || !single) return DWF_EINVAL;
    DWF_TRY(mrhs_ok(c, nrhs));
    if (j < 0 || j >= nrhs) { c->err = "mrhs: system index out of range"; return DWF_EINVAL; }
    const size_t chunk = half_bytes(c->g, prec) / c->g.ntiles;
    DWF_CUDA_CHECK(c, cudaMemcpy2DAsync(single, chunk, (const char*)batched + j * chunk, chunk * nrhs, chunk, c->g.ntiles,
                                        cudaMemcpyDeviceToDevice, c->stream));
    return DWF_OK;
}

dwf_status dwf_dhop_mrhs(dwf_ctx* c, void* out, const void* in, int nrhs, dwf_parity out_parity, int dagger, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out || !in || out == in || out_parity == DWF_FULL) { c->err = "dhop_mrhs: null / aliased pointers or FULL parity"; return DWF_EINVAL; }
    DWF_TRY(mrhs_ok(c, nrhs));
    BatchGuard bg(c, nrhs);
    return launch_dhop(c, out, in, out_parity, dagger, prec);
}

dwf_status dwf_mpc_mrhs(dwf_ctx* c, void* out, const void* in, int nrhs, int dagger, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out || !in || out == in) { c->err = "mpc_mrhs: null or aliased pointers"; return DWF_EINVAL; }
    DWF_TRY(mrhs_ok(c, nrhs));
    if (nrhs > 1) DWF_TRY(wsm_reserve(c, nrhs));
    BatchGuard bg(c, nrhs);
    return mpc_apply(c, out, in, dagger, prec, -1);
}

dwf_status dwf_mdagm_mrhs(dwf_ctx* c, void* out, const void* in, int nrhs, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out || !in || out == in) { c->err = "mdagm_mrhs: null or aliased pointers"; return DWF_EINVAL; }
    DWF_TRY(mrhs_ok(c, nrhs));
    if (nrhs > 1) DWF_TRY(wsm_reserve(c, nrhs));
    BatchGuard bg(c, nrhs);
    return mdagm_apply(c, out, in, prec);
}

dwf_status dwf_cg_mrhs(dwf_ctx* c, void* x, const void* b, int nrhs, double tol, int max_iter, dwf_cg_mode mode, int use_guess,
                       dwf_cg_info* info) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!x || !b || x == b || !info || tol <= 0.0 || max_iter < 0) { c->err = "cg_mrhs: bad arguments"; return DWF_EINVAL; }
    DWF_TRY(mrhs_ok(c, nrhs));
    memset(info, 0, sizeof(*info) * nrhs);
    if (nrhs > 1) DWF_TRY(wsm_reserve(c, nrhs));
    BatchGuard bg(c, nrhs);
    const long long l0 = c->launches;
    const double t0 = now_s();
    dwf_status st = (mode == DWF_CG_MIXED) ? cg_mixed(c, x, b, tol, max_iter, use_guess, info)
                                           : cg_f64(c, x, b, tol, max_iter, use_guess, info);
    cudaStreamSynchronize(c->stream);
    for (int j = 0; j < nrhs; ++j) {
        info[j].seconds = now_s() - t0;
        info[j].launches = (int)(c->launches - l0);
    }
    if (st == DWF_ENOTCONV) c->err = "cg_mrhs: max_iter reached";
    return st;
}

dwf_status dwf_multishift_cg(dwf_ctx* c, void* xv, const void* b, const double* shifts, int nshift, double tol, int max_iter,
                             dwf_cg_info* info, double* resid_true) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    dwf_cg_info local;
    if (!info) info = &local;
    memset(info, 0, sizeof(*info));
    if (!xv || !b || xv == b || !shifts || nshift < 1 || nshift > 16 || tol <= 0.0 || max_iter < 0 || shifts[0] < 0.0) {
        c->err = "multishift_cg: bad arguments";
        return DWF_EINVAL;
    }
    for (int i = 1; i < nshift; ++i)
        if (shifts[i] < shifts[i - 1]) { c->err = "multishift_cg: shifts must ascend"; return DWF_EINVAL; }
    const long long l0 = c->launches;
    const double t0 = now_s();
    const int P = DWF_F64;
    const size_t hb = half_bytes(c->g, P), n = half_reals(c);
    if (c->ms_p_bytes < hb * nshift) {
        if (c->ms_p) cudaFree(c->ms_p);
        c->ms_p = nullptr; c->ms_p_bytes = 0;
        if (cudaMalloc(&c->ms_p, hb * nshift) != cudaSuccess) { cudaGetLastError(); c->err = "cudaMalloc(multishift) failed"; return DWF_ENOMEM; }
        c->ms_p_bytes = hb * nshift;
    }
    char* x = (char*)xv;
    char* p = (char*)c->ms_p;
    void *r, *q, *z;
    DWF_TRY(ws_get(c, P, 2, &r));
    DWF_TRY(ws_get(c, P, 4, &q));
    DWF_TRY(ws_get(c, P, 5, &z));
    double bn2;
    DWF_TRY(norm2_host(c, b, P, &bn2));
    DWF_CUDA_CHECK(c, cudaMemsetAsync(x, 0, hb * nshift, c->stream));
    if (bn2 == 0.0) {
        if (resid_true) for (int i = 0; i < nshift; ++i) resid_true[i] = 0.0;
        return DWF_OK;
    }
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(r, b, hb, cudaMemcpyDeviceToDevice, c->stream));
    for (int i = 0; i < nshift; ++i) DWF_CUDA_CHECK(c, cudaMemcpyAsync(p + i * hb, b, hb, cudaMemcpyDeviceToDevice, c->stream));
    // The scalar recurrences (alpha, beta, zeta_i and the update coefficients) live on the device (MsState); the stopping
    // test is the CG's (cg_conv[0]) and the host runs one iteration ahead of the residual it has read, exactly as in
    // cg_iterate: no stream synchronisation inside the loop.
    const double s0 = shifts[0], target = tol * tol * bn2;
    {
        MsState h;
        memset(&h, 0, sizeof(h));
        h.n = nshift; h.s0 = s0; h.cc = bn2; h.p0n2 = bn2; h.alpha_old = 1.0; h.beta_old = 0.0;
        for (int i = 0; i < nshift; ++i) { h.delta[i] = shifts[i] - s0; h.zeta[i] = h.zeta_old[i] = 1.0; }
        if (!c->ms_state && cudaMalloc(&c->ms_state, sizeof(MsState)) != cudaSuccess) { cudaGetLastError(); c->err = "cudaMalloc(multishift state) failed"; return DWF_ENOMEM; }
        DWF_CUDA_CHECK(c, cudaMemcpyAsync(c->ms_state, &h, sizeof(h), cudaMemcpyHostToDevice, c->stream));
        CgRun run;
        run.n = 1; run.target[0] = target; run.c[0] = bn2;
        DWF_TRY(cg_upload_state(c, run, SLOT_C));          // cg_target[0], cg_conv[0] = -1 (synchronises: h may go out of scope)
    }
    double cc = bn2;
    int iters = 0, k = 0, decided = 0;
    bool done = (cc <= target);
    auto decide = [&](int it, dwf_status* st) -> bool {
        *st = DWF_OK;
        if (cudaEventSynchronize(c->cg_ev[it % CG_RING]) != cudaSuccess) { c->err = "cudaEventSynchronize failed"; *st = DWF_ECUDA; return true; }
        const double cn = c->cn_ring[(size_t)(it % CG_RING) * MAXR];
        if (!(cn == cn)) { c->err = "multishift_cg: NaN residual"; *st = DWF_ECUDA; return true; }
        cc = cn;
        iters = it;
        decided = it;
        return cn <= target;
    };
    dwf_status lst = DWF_OK;
    while (!done && k < max_iter) {
        ++k;
        // q = Mpc p_0 (|q|^2 -> SLOT_D), z = Mpc^dag q;  d = <p_0, (A + s0) p_0> = |q|^2 + s0 |p_0|^2
        DWF_TRY(mpc_apply(c, q, p, 0, P, SLOT_D));
        DWF_TRY(mpc_apply(c, z, q, 1, P, -1));
        DWF_TRY(launch_ms_r(c, r, z, p, n, SLOT_D, SLOT_CN, k));               // alpha, zeta'; r -= alpha (z + s0 p_0); |r|^2, test
        DWF_CUDA_CHECK(c, cudaMemcpyAsync(c->cn_ring + (size_t)(k % CG_RING) * MAXR, c->scalars + (size_t)SLOT_CN * MAXR, sizeof(double),
                                          cudaMemcpyDeviceToHost, c->stream));
        DWF_CUDA_CHECK(c, cudaEventRecord(c->cg_ev[k % CG_RING], c->stream));
        DWF_TRY(launch_ms_update(c, x, p, r, n, SLOT_CN, SLOT_T1, k));         // beta; x_i += .. p_i ; p_i = .. ; |p_0|^2
        if (k >= 2 && decide(k - 1, &lst)) { done = true; break; }
    }
    if (lst != DWF_OK) return lst;
    while (!done && decided < k) {
        done = decide(decided + 1, &lst);
        if (lst != DWF_OK) return lst;
    }
    info->iters_total = iters;
    info->resid_iter = std::sqrt(cc / bn2);
    // true residuals: b - (A + s_i) x_i
    double worst = 0.0;
    for (int i = 0; i < nshift; ++i) {
        DWF_TRY(mdagm_apply(c, z, x + i * hb, P));
        DWF_TRY(launch_sub(c, q, b, z, P, n));
        DWF_TRY(launch_axpy(c, q, x + i * hb, -shifts[i], P, n));
        double rn2;
        DWF_TRY(norm2_host(c, q, P, &rn2));
        const double rt = std::sqrt(rn2 / bn2);
        if (resid_true) resid_true[i] = rt;
        if (rt > worst) worst = rt;
    }
    info->resid_true = worst;
    cudaStreamSynchronize(c->stream);
    info->seconds = now_s() - t0;
    info->launches = (int)(c->launches - l0);
    if (cc > target) { c->err = "multishift_cg: max_iter reached"; return DWF_ENOTCONV; }
    return DWF_OK;
}

dwf_status dwf_chebyshev(dwf_ctx* c, void* out, const void* in, double lo, double hi, int order, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out || !in || out == in || !(hi > lo) || order < 0) { c->err = "chebyshev: bad arguments"; return DWF_EINVAL; }
    const size_t hb = half_bytes(c->g, prec), n = half_reals(c);
    const double s = 2.0 / (hi - lo), o = -(hi + lo) / (hi - lo);
    if (order == 0) {
        DWF_CUDA_CHECK(c, cudaMemcpyAsync(out, in, hb, cudaMemcpyDeviceToDevice, c->stream));
        return DWF_OK;
    }
    void *ta, *tb, *av;
    DWF_TRY(ws_get(c, prec, 6, &av));
    DWF_TRY(ws_get(c, prec, 7, &ta));
    DWF_TRY(ws_get(c, prec, 8, &tb));
    // t_1 = s A in + o in
    DWF_TRY(mdagm_apply(c, av, in, prec));
    void* t1 = (order == 1) ? out : ta;
    DWF_TRY(launch_lincomb3(c, t1, av, in, in, s, o, 0.0, prec, n));
    const void* tkm1 = in;          // t_{k-1}
    void* tk = t1;                  // t_k
    for (int k = 1; k < order; ++k) {
        // t_{k+1} = 2 s A t_k + 2 o t_k - t_{k-1}, written over the buffer that is free (never over `in`)
        DWF_TRY(mdagm_apply(c, av, tk, prec));
        void* dst = (k + 1 == order) ? out : ((tk == ta) ? tb : ta);
        DWF_TRY(launch_lincomb3(c, dst, av, tk, tkm1, 2.0 * s, 2.0 * o, -1.0, prec, n));
        tkm1 = tk;
        tk = dst;
    }
    return DWF_OK;
}

dwf_status dwf_solve(dwf_ctx* c, void* psi, const void* eta, double tol, int max_iter, dwf_cg_mode mode, dwf_cg_info* info) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    dwf_cg_info local;
    if (!info) info = &local;
    memset(info, 0, sizeof(*info));
    if (!psi || !eta || psi == eta || tol <= 0.0 || max_iter < 0) { c->err = "solve: bad arguments"; return DWF_EINVAL; }
    const long long l0 = c->launches;
    const double t0 = now_s();
    const int P = DWF_F64;
    const size_t hb = half_bytes(c->g, P);
    const void* eta_e = eta;
    const void* eta_o = (const char*)eta + hb;
    void* psi_e = psi;
    void* psi_o = (char*)psi + hb;
    void *t1, *t2, *src, *rhs;
    DWF_TRY(ws_get(c, P, 0, &t1));
    DWF_TRY(ws_get(c, P, 1, &t2));
    DWF_TRY(ws_get(c, P, 8, &src));
    DWF_TRY(ws_get(c, P, 9, &rhs));
    // src = eta_o - Moe Mee^-1 eta_e = eta_o + 1/2 Dhop_o A Mee^-1 eta_e
    DWF_TRY(launch_op5(c, t1, eta_e, OP_A_MEEINV, nullptr, -1, 0.0, P, -1));
    DWF_TRY(launch_dhop(c, t2, t1, DWF_ODD, 0, P));
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(src, eta_o, hb, cudaMemcpyDeviceToDevice, c->stream));
    DWF_TRY(launch_axpy(c, src, t2, 0.5, P, half_reals(c)));
    DWF_TRY(mpc_apply(c, rhs, src, 1, P, -1));
    dwf_status st = (mode == DWF_CG_MIXED) ? cg_mixed(c, psi_o, rhs, tol, max_iter, 0, info)
                                           : cg_f64(c, psi_o, rhs, tol, max_iter, 0, info);
    if (st != DWF_OK && st != DWF_ENOTCONV) return st;
    // psi_e = Mee^-1 (eta_e - Meo psi_o) = Mee^-1 (eta_e + 1/2 Dhop_e A psi_o)
    DWF_TRY(launch_op5(c, t1, psi_o, OP_A, nullptr, -1, 0.0, P, -1));
    DWF_TRY(launch_dhop(c, t2, t1, DWF_EVEN, 0, P));
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(t1, eta_e, hb, cudaMemcpyDeviceToDevice, c->stream));
    DWF_TRY(launch_axpy(c, t1, t2, 0.5, P, half_reals(c)));
    DWF_TRY(launch_op5(c, psi_e, t1, OP_MEEINV, nullptr, -1, 0.0, P, -1));
    // |eta - M psi| / |eta|
    void *me, *mo;
    DWF_TRY(ws_get(c, P, 2, &me));
    DWF_TRY(ws_get(c, P, 3, &mo));
    double en2 = 0, rn2 = 0, v;
    for (int p = 0; p < 2; ++p) {
        const void* in_p = (const char*)psi + p * hb;
        const void* in_q = (const char*)psi + (1 - p) * hb;
        const void* e_p = (const char*)eta + p * hb;
        DWF_TRY(launch_op5(c, t1, in_q, OP_A, nullptr, -1, 0.0, P, -1));
        DWF_TRY(launch_dhop(c, t2, t1, p, 0, P));
        DWF_TRY(launch_op5(c, me, in_p, OP_MEE, t2, -1, -0.5, P, -1));
        DWF_TRY(launch_sub(c, mo, e_p, me, P, half_reals(c)));
        DWF_TRY(norm2_host(c, mo, P, &v)); rn2 += v;
        DWF_TRY(norm2_host(c, e_p, P, &v)); en2 += v;
    }
    info->resid_full = (en2 > 0) ? std::sqrt(rn2 / en2) : 0.0;
    cudaStreamSynchronize(c->stream);
    info->seconds = now_s() - t0;
    info->launches = (int)(c->launches - l0);
    return st;
}

// ---- domain / boundary projectors and the boundary operators R, R^-1 (eqs. 8-14)
static dwf_status boundary_geometry_ok(dwf_ctx* c) {
    bool any = false;
    for (int mu = 0; mu < 4; ++mu)
        if (c->cut[mu] > 0) {
            any = true;
            if ((c->g.L[mu] / c->cut[mu]) & 1) { c->err = "boundary operators need an even number of Dirichlet blocks in every cut direction"; return DWF_EINVAL; }
        }
    if (!any) { c->err = "boundary operators need a Dirichlet cut (dwf_create dirichlet_cut)"; return DWF_EINVAL; }
    return DWF_OK;
}

dwf_status dwf_domain_project(dwf_ctx* c, void* out, const void* in, int which, dwf_prec prec) {
    DeviceGuard _dev(c);
    if (!c || !out || !in || which < 0 || which > 2) return DWF_EINVAL;
    DWF_TRY(boundary_geometry_ok(c));
    const size_t hb = half_bytes(c->g, prec);
    for (int p = 0; p < 2; ++p) DWF_TRY(launch_domain_project(c, (char*)out + p * hb, (const char*)in + p * hb, p, which, prec));
    return DWF_OK;
}

namespace {
struct LinkGuard {      // the uncut link set is only ever visible inside one ABI call
    dwf_ctx* c;
    explicit LinkGuard(dwf_ctx* cc) : c(cc) {}
    ~LinkGuard() { select_links(c, false); }
};
// out = P_to M_uncut P_from in  (the zero-padded boundary blocks of eq. 4: from = 0, to = 1 is D_dbar_hat; from = 1, to = 0 D_d_hat)
dwf_status boundary_block(dwf_ctx* c, void* out, const void* in, void* tmp, int from, int to) {
    DWF_TRY(dwf_domain_project(c, tmp, in, from, DWF_F64));
    select_links(c, true);
    DWF_TRY(m_apply(c, out, tmp, 0, DWF_F64));
    select_links(c, false);
    return dwf_domain_project(c, out, out, to, DWF_F64);
}
}  // namespace

dwf_status dwf_boundary_op(dwf_ctx* c, void* out, const void* in, int inverse, double tol, int max_iter, dwf_cg_mode mode,
                           dwf_cg_info* info) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    dwf_cg_info local;
    if (!info) info = &local;
    memset(info, 0, sizeof(*info));
    if (!out || !in || out == in || tol <= 0.0 || max_iter < 0) { c->err = "boundary_op: bad arguments"; return DWF_EINVAL; }
    DWF_TRY(boundary_geometry_ok(c));
    const double t0 = now_s();
    const long long l0 = c->launches;
    const size_t fb = 2 * half_bytes(c->g, DWF_F64);
    if (c->bnd_ws_bytes < 2 * fb) {
        if (c->bnd_ws) cudaFree(c->bnd_ws);
        c->bnd_ws = nullptr; c->bnd_ws_bytes = 0;
        if (cudaMalloc(&c->bnd_ws, 2 * fb) != cudaSuccess) { cudaGetLastError(); c->err = "cudaMalloc(boundary workspace) failed"; return DWF_ENOMEM; }
        c->bnd_ws_bytes = 2 * fb;
    }
    void* u = c->bnd_ws;
    void* v = (char*)c->bnd_ws + fb;
    LinkGuard guard(c);
    dwf_cg_info si;
    dwf_status st, worst = DWF_OK;
    int iters = 0;
    double rfull = 0.0;
    DWF_TRY(boundary_block(c, u, in, v, 0, 1));                         // u = D_dbar_hat phi            (on Omegabar)
    if (inverse) {
        select_links(c, true);                                          // v = D^-1 u                    (eq. 13)
        st = dwf_solve(c, v, u, tol, max_iter, mode, &si);
        select_links(c, false);
        if (st != DWF_OK && st != DWF_ENOTCONV) return st;
        if (st != DWF_OK) worst = st;
        iters += si.iters_total; rfull = si.resid_full;
    } else {
        st = dwf_solve(c, v, u, tol, max_iter, mode, &si);              // v = D_Ob^-1 u  (the cut operator is D_O + D_Ob)
        if (st != DWF_OK && st != DWF_ENOTCONV) return st;
        if (st != DWF_OK) worst = st;
        iters += si.iters_total; rfull = si.resid_full;
        DWF_TRY(boundary_block(c, u, v, out, 1, 0));                    // u = D_d_hat v                 (on Omega; out as scratch)
        st = dwf_solve(c, v, u, tol, max_iter, mode, &si);              // v = D_O^-1 u                  (eq. 9)
        if (st != DWF_OK && st != DWF_ENOTCONV) return st;
        if (st != DWF_OK) worst = st;
        iters += si.iters_total; rfull = std::fmax(rfull, si.resid_full);
    }
    DWF_TRY(dwf_domain_project(c, u, v, 2, DWF_F64));                   // P v
    DWF_TRY(dwf_domain_project(c, out, in, 2, DWF_F64));                // P phi
    DWF_TRY(launch_axpy(c, out, u, -1.0, DWF_F64, 2 * half_reals(c)));  // out = P phi - P v
    cudaStreamSynchronize(c->stream);
    info->iters_total = iters;
    info->resid_full = rfull;
    info->seconds = now_s() - t0;
    info->launches = (int)(c->launches - l0);
    return worst;
}

dwf_status dwf_dhop_host(dwf_ctx* c, void* out_host, const void* in_host, dwf_parity out_parity, int dagger, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out_host || !in_host) return DWF_EINVAL;
    const size_t nb = dwf_field_bytes(c, prec, out_parity);
    void *canon, *nat;
    DWF_TRY(stage_get(c, 0, nb, &canon));
    DWF_TRY(stage_get(c, 1, 2 * nb, &nat));
    void* nat_in = nat;
    void* nat_out = (char*)nat + nb;
    const dwf_parity in_par = (out_parity == DWF_FULL) ? DWF_FULL : (out_parity == DWF_EVEN ? DWF_ODD : DWF_EVEN);
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(canon, in_host, nb, cudaMemcpyHostToDevice, c->stream));
    DWF_TRY(launch_pack(c, nat_in, canon, prec, in_par, false));
    DWF_TRY(dwf_dhop(c, nat_out, nat_in, out_parity, dagger, prec));
    DWF_TRY(launch_pack(c, nat_out, canon, prec, out_parity, true));
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(out_host, canon, nb, cudaMemcpyDeviceToHost, c->stream));
    DWF_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return DWF_OK;
}

dwf_status dwf_mdagm_host(dwf_ctx* c, void* out_host, const void* in_host, dwf_prec prec) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!out_host || !in_host) return DWF_EINVAL;
    const size_t nb = dwf_field_bytes(c, prec, DWF_ODD);
    void *canon, *nat;
    DWF_TRY(stage_get(c, 0, nb, &canon));
    DWF_TRY(stage_get(c, 1, 2 * nb, &nat));
    void* nat_in = nat;
    void* nat_out = (char*)nat + nb;
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(canon, in_host, nb, cudaMemcpyHostToDevice, c->stream));
    DWF_TRY(launch_pack(c, nat_in, canon, prec, DWF_ODD, false));
    DWF_TRY(mdagm_apply(c, nat_out, nat_in, prec));
    DWF_TRY(launch_pack(c, nat_out, canon, prec, DWF_ODD, true));
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(out_host, canon, nb, cudaMemcpyDeviceToHost, c->stream));
    DWF_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return DWF_OK;
}

dwf_status dwf_cg_host(dwf_ctx* c, void* x_host, const void* b_host, double tol, int max_iter, dwf_cg_mode mode,
                       dwf_cg_info* info) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!x_host || !b_host) return DWF_EINVAL;
    const double t0 = now_s();
    const long long l0 = c->launches;
    const size_t nb = dwf_field_bytes(c, DWF_F64, DWF_ODD);
    void *canon, *nat;
    DWF_TRY(stage_get(c, 0, nb, &canon));
    DWF_TRY(stage_get(c, 1, 2 * nb, &nat));
    void* nat_b = nat;
    void* nat_x = (char*)nat + nb;
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(canon, b_host, nb, cudaMemcpyHostToDevice, c->stream));
    DWF_TRY(launch_pack(c, nat_b, canon, DWF_F64, DWF_ODD, false));
    dwf_status st = dwf_cg(c, nat_x, nat_b, tol, max_iter, mode, 0, info);
    if (st != DWF_OK && st != DWF_ENOTCONV) return st;
    DWF_TRY(launch_pack(c, nat_x, canon, DWF_F64, DWF_ODD, true));
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(x_host, canon, nb, cudaMemcpyDeviceToHost, c->stream));
    DWF_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (info) { info->seconds = now_s() - t0; info->launches = (int)(c->launches - l0); }
    return st;
}

dwf_status dwf_solve_host(dwf_ctx* c, void* psi_host, const void* eta_host, double tol, int max_iter, dwf_cg_mode mode,
                          dwf_cg_info* info) {
    DeviceGuard _dev(c);
    DWF_TRY(need_gauge(c));
    if (!psi_host || !eta_host) return DWF_EINVAL;
    const double t0 = now_s();
    const long long l0 = c->launches;
    const size_t nb = dwf_field_bytes(c, DWF_F64, DWF_FULL);
    void *canon, *nat;
    DWF_TRY(stage_get(c, 0, nb, &canon));
    DWF_TRY(stage_get(c, 1, 2 * nb, &nat));
    void* nat_eta = nat;
    void* nat_psi = (char*)nat + nb;
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(canon, eta_host, nb, cudaMemcpyHostToDevice, c->stream));
    DWF_TRY(launch_pack(c, nat_eta, canon, DWF_F64, DWF_FULL, false));
    dwf_status st = dwf_solve(c, nat_psi, nat_eta, tol, max_iter, mode, info);
    if (st != DWF_OK && st != DWF_ENOTCONV) return st;
    DWF_TRY(launch_pack(c, nat_psi, canon, DWF_F64, DWF_FULL, true));
    DWF_CUDA_CHECK(c, cudaMemcpyAsync(psi_host, canon, nb, cudaMemcpyDeviceToHost, c->stream));
    DWF_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (info) { info->seconds = now_s() - t0; info->launches = (int)(c->launches - l0); }
    return st;
}

long long dwf_launch_count(const dwf_ctx* c) { return c ? c->launches : 0; }
const char* dwf_last_error(const dwf_ctx* c) { return c ? c->err.c_str() : "null context"; }

}  // extern "C"
