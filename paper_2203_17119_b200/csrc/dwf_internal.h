// Internal declarations of the dwf_b200 library (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../../include/dwf.h"

namespace dwf {

// ---------------------------------------------------------------------------------------------
// Native layout.  One parity of a field:
//     vec index = ((tile * Ls + s) * K + k) * TS + lane          (16-byte vectors)
// K = 24/VW vectors per spinor (VW = 4 floats or 2 doubles), TS = sites of one parity in a tile.
// tile = ((it*NT[2] + iz)*NT[1] + iy)*NT[0] + ix ; lane = ((tt*T[2] + tz)*T[1] + ty)*(T[0]/2) + tx/2.
// Gauge, per OUTPUT parity: vec index = ((tile * 8 + leg) * KG + kg) * TS + lane, leg = 2*mu + dir,
// dir 0: W = U_mu(x) (forward), dir 1: W = U_mu(x-mu)^dag (backward); 12 (rows 0,1) or 18 reals.
// ---------------------------------------------------------------------------------------------
// Batched ("multi right-hand side") fields: N systems that share one gauge field are stored as ONE
// native field whose fifth dimension is N*Ls long, slice index rhs*Ls + s:
//     vec index = (((tile * N + rhs) * Ls + s) * K + k) * TS + lane
// The Dhop kernels do not look at s, so they run on such a field with Ls := N*Ls and load the links of a tile once for all
// N*Ls slices; the column kernels and the Dhop epilogue take N and the physical Ls (the -mf walls sit at s = 0, Ls-1 of
// every system).  Scalar slot `slot` of system `rhs` is scalars[slot * MAXR + rhs].
constexpr int MAXR = 16;

struct Geom {
    int L[4];    // lattice extents
    int T[4];    // tile extents
    int NT[4];   // tiles per direction
    int TS;      // sites of one parity per tile
    int ntiles;  // number of tiles
    int Vh;      // sites of one parity  (= ntiles*TS)
    int Ls;
    int antiperiodic_t;
    int swz;     // lane order: y rows XOR-rotated by tz (dwf_layout.cuh); set per precision by geom_prec()
};

// 5-D coefficient tables: out_s = sum_s' Tp[s][s'] in_s' on P+ components (spin 0,1), Tm on P- (spin 2,3)
struct Table5 {
    double p[32 * 32];
    double m[32 * 32];
};

enum Op5 { OP_A = 0, OP_ADAG, OP_MEE, OP_MEEDAG, OP_MEEINV, OP_MEEINVDAG,
           OP_A_MEEINV,        // A * Mee^-1            (middle of Mpc)
           OP_MEEINVDAG_ADAG,  // Mee^-dag * A^dag      (middle of Mpc^dag)
           OP5_COUNT };

// device-resident scalar state of the multishift CG (dwf_blas.cu): zeta recurrences of every shift, the base system's
// alpha / beta / |r|^2 / |p_0|^2 and the coefficients the vector kernels read
struct MsState {
    int n;
    double s0, cc, p0n2, alpha, alpha_old, beta_old;
    double delta[16], zeta[16], zeta_old[16], znew[16], ax[16], zr[16], bp[16];
};

struct DevTables {           // device copies, [OP5_COUNT][2][Ls*Ls]
    double* d64 = nullptr;
    float* d32 = nullptr;
};

}  // namespace dwf

struct dwf_ctx {
    dwf::Geom g;
    double M5, mf, b5, c5;
    int cut[4];
    int compress12 = 1;
    int tile_opt[4] = {0, 0, 0, 0};
    int dhop_kernel = 0;   // 0 = auto (TMA kernel for 4^4 tiles, else cp.async tile kernel, else generic), 1 = generic, 2 = cp.async tile kernel
    int fuse = 1;          // Mpc / CG through the Dhop kernel's fused 5-D epilogues when the TMA kernel applies (0: separate op5 kernels)
    int dhop_dynamic = 1;  // TMA kernel tile scheduling: 1 global in-order queue (default), 0 static round-robin (same results: every reduction is per tile)
    void* tma = nullptr;   // dwf::TmaState (dwf_dhop_tma.cu), built at dwf_set_gauge for 4^4 tiles
    // tables of the pipelined Dhop kernel (dwf_dhop_pipe.cu), built at dwf_set_gauge
    uint16_t* pipe_nbslot[2] = {nullptr, nullptr};      // [precision]: the two precisions differ in lane order
    int16_t* pipe_slot_dir[2] = {nullptr, nullptr};
    uint16_t* pipe_slot_lane[2] = {nullptr, nullptr};
    int swz64 = 0;         // fp64 native fields use the XOR-rotated lane order (4^4 tiles); fp32 fields never do
    int pipe_nslot = 0;
    double inner_tol = 1e-4;
    int max_restarts = 20;
    cudaStream_t stream = nullptr;
    int device = 0;        // CUDA device the context was created on; every ABI call runs with it current (DeviceGuard)
    int num_sms = 148;     // cudaDevAttrMultiProcessorCount of that device (dwf_create): grid sizes of the streaming kernels
    bool gauge_set = false;
    bool geom_frozen = false;
    // gauge copies [parity]
    void* W64[2] = {nullptr, nullptr};
    void* W32[2] = {nullptr, nullptr};
    size_t wbytes64 = 0, wbytes32 = 0;
    // second link set WITHOUT the Dirichlet cut (built when a cut is configured): the boundary operators of eqs. 8-14 need
    // D and D_Omega + D_Omegabar on the same gauge field.  select_links() swaps it with W64 / W32.
    void* W64u[2] = {nullptr, nullptr};
    void* W32u[2] = {nullptr, nullptr};
    bool links_uncut = false;
    void* bnd_ws = nullptr;      // boundary operators: two FULL fp64 fields
    size_t bnd_ws_bytes = 0;
    dwf::Table5 tab[dwf::OP5_COUNT];
    dwf::DevTables dtab;
    // solver workspace: 10 half fields per precision, allocated at dwf_set_gauge (ws_alloc_all, dwf_api.cu)
    void* ws64[10] = {};
    void* ws32[10] = {};
    dwf::MsState* ms_state = nullptr;   // multishift CG: device-resident scalar recurrences
    void* ms_p = nullptr;        // multishift CG: search directions of all shifts
    size_t ms_p_bytes = 0;
    double* partials = nullptr;  // per-block reduction partials
    int npartials = 0;
    double* scalars = nullptr;   // device scalars [NSLOTS][MAXR]
    double* scalars_host = nullptr;  // pinned, same shape
    // device-side stopping test of the CG (one entry per right-hand side): cg_target = tol^2 |b|^2, cg_conv = first
    // iteration with |r|^2 <= target (-1: none yet).  The host runs one iteration ahead of what it has read back.
    double* cg_target = nullptr;     // device [MAXR]
    int* cg_conv = nullptr;          // device [MAXR]
    double* cn_ring = nullptr;       // pinned [CG_RING][MAXR]: |r|^2 of the last iterations
    cudaEvent_t cg_ev[4] = {nullptr, nullptr, nullptr, nullptr};
    // workspace of the batched (multi right-hand side) calls: NWS fields of mrhs_cap systems per precision
    void* wsm64[10] = {};
    void* wsm32[10] = {};
    int mrhs_cap = 0;
    int nrhs_cur = 1;      // right-hand sides of the call in progress (1 outside the *_mrhs entry points)
    void* stage_dev[2] = {nullptr, nullptr};  // staging for *_host calls
    size_t stage_bytes[2] = {0, 0};
    long long launches = 0;
    // optional per-launch CUDA-event timing of the Dhop kernel ("time_dhop" option; bench.py's roofline)
    int time_dhop = 0;
    std::vector<cudaEvent_t> ev;     // pairs (start, stop)
    int ev_used = 0;
    double dhop_ms = 0.0;
    double dhop_bytes = 0.0;     // algorithmic bytes of the timed launches
    long long dhop_timed = 0;
    std::string err;
};

namespace dwf {

// geometry as seen by fields of one precision: fp64 fields of 4^4 tiles are stored in the XOR-rotated lane order that makes
// the fp64 Dhop kernel's shared-memory accesses conflict-free; fp32 fields keep the plain order (its kernel has no
// registers left for the extra face gathers that order needs).  dwf_convert and x64 += e32 permute the lanes.
inline Geom geom_prec(const dwf_ctx* c, int prec, int nrhs = 1) {
    Geom g = c->g;
    g.swz = (prec == DWF_F64) ? c->swz64 : 0;
    g.Ls *= nrhs;          // batched field: the Dhop kernels see one long fifth dimension
    return g;
}

inline size_t half_vecs(const Geom& g, int prec) { return (size_t)g.Vh * g.Ls * (prec == DWF_F64 ? 12 : 6); }
inline size_t half_bytes(const Geom& g, int prec) { return half_vecs(g, prec) * 16; }

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: one bit per device ordinal and kernel instantiation
inline bool attr_needed(unsigned long long& done_mask, int device) {
    const unsigned long long bit = 1ull << (device & 63);
    if (done_mask & bit) return false;
    done_mask |= bit;
    return true;
}

// makes the context's device current for the duration of an ABI call and restores the caller's device afterwards
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const dwf_ctx* c) {
        if (!c) return;
        int cur = 0;
        if (cudaGetDevice(&cur) == cudaSuccess && cur != c->device && cudaSetDevice(c->device) == cudaSuccess) prev = cur;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

#define DWF_CUDA_CHECK(ctx, expr)                                                            \
    do {                                                                                     \
        cudaError_t _e = (expr);                                                             \
        if (_e != cudaSuccess) {                                                             \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(_e);                 \
            return DWF_ECUDA;                                                                \
        }                                                                                    \
    } while (0)

// kernels / launchers (one translation unit each)
dwf_status launch_dhop(dwf_ctx* c, void* out, const void* in, int out_parity, int dagger, int prec);
// out = T[op1] x (+ yscale*y if y && op2<0 | + yscale*T[op2] y if y && op2>=0); norm_slot>=0: |out|^2 -> scalars[slot]
dwf_status launch_op5(dwf_ctx* c, void* out, const void* x, int op1, const void* y, int op2, double yscale,
                      int prec, int norm_slot);
dwf_status launch_gauge_prep(dwf_ctx* c, const double* Ucanon);
void select_links(dwf_ctx* c, bool uncut);   // which link set the operators see (must be back on `cut` when an ABI call returns)
// out = P in on one half field of `parity`: which = 0 P_Omega, 1 P_Omegabar, 2 the boundary projector P_dbar (fp64 or fp32)
dwf_status launch_domain_project(dwf_ctx* c, void* out, const void* in, int parity, int which, int prec);
dwf_status launch_pack(dwf_ctx* c, void* native, const void* canon, int prec, int parity, bool unpack);
dwf_status launch_convert(dwf_ctx* c, void* dst, int dprec, const void* src, int sprec, size_t nhalf_fields);
// BLAS-1 on native half fields; scalar slots index c->scalars
dwf_status launch_norm2(dwf_ctx* c, const void* v, int prec, size_t nreal, int slot);
dwf_status launch_cg_update(dwf_ctx* c, void* x, void* r, const void* p, const void* z, int prec, size_t nreal,
                            int slot_c, int slot_d, int slot_cn, int iter);  // x+=a p; r-=a z; cn=|r|^2, a=c/d (iter: stopping test)
dwf_status launch_xpay(dwf_ctx* c, void* p, const void* r, int prec, size_t nreal, int slot_cn, int slot_c);  // p=r+(cn/c)p
dwf_status launch_axpy(dwf_ctx* c, void* y, const void* x, double a, int prec, size_t nreal);  // y += a x
dwf_status launch_sub(dwf_ctx* c, void* out, const void* a, const void* b, int prec, size_t nreal);  // out = a - b
dwf_status launch_add_f32_to_f64(dwf_ctx* c, void* x64, const void* e32, size_t unused);  // x += (double)e, half field
// multishift CG: alpha / zeta recurrences from scalars[slot_d] and c->ms_state, then r -= alpha (z + s0 p_0), |r|^2 -> slot (+ test)
dwf_status launch_ms_r(dwf_ctx* c, void* r, const void* z, const void* p0, size_t nreal, int slot_d, int slot, int iter);
// beta and the update coefficients from scalars[slot_cn], then all shifts: x_i += .., p_i = ..; |p_0|^2 -> slot and state
dwf_status launch_ms_update(dwf_ctx* c, void* x, void* p, const void* r, size_t nreal, int slot_cn, int slot, int iter);
dwf_status launch_lincomb3(dwf_ctx* c, void* out, const void* x, const void* y, const void* z, double a, double b, double cc,
                           int prec, size_t nreal);   // out = a x + b y + cc z
dwf_status ensure_partials(dwf_ctx* c, int n);
dwf_status launch_reduce(dwf_ctx* c, int n, int slot, int iter = 0);   // iter > 0: also the CG stopping test of that iteration
void build_tables(dwf_ctx* c);
dwf_status pipe_tables_upload(dwf_ctx* c);
void pipe_tables_free(dwf_ctx* c);
dwf_status launch_dhop_pipe(dwf_ctx* c, void* out, const void* in, int out_parity, int dagger, int prec, bool* handled);
dwf_status tma_state_build(dwf_ctx* c);
void tma_state_free(dwf_ctx* c);
dwf_status launch_dhop_tma(dwf_ctx* c, void* out, const void* in, int out_parity, int dagger, int prec, bool* handled);
// Dhop with the fused last step of Mpc (dwf_dhop_tma.cu): out = Mee xin + scale Dhop in, norm_slot >= 0: |out|^2
enum { EPI_NONE = 0, EPI_FINAL = 1 };
bool dhop_fused_available(const dwf_ctx* c);
dwf_status launch_dhop_fused(dwf_ctx* c, void* out, const void* in, int out_parity, int prec, const void* xin, double scale,
                             int norm_slot);
// r -= (sc[slot_c]/sc[slot_d]) (Mee^dag q + yscale A^dag d); |r|^2 -> scalars[norm_slot]   (dwf_fived.cu)
dwf_status launch_cg_r(dwf_ctx* c, void* r, const void* q, const void* d, double yscale, int prec, int slot_c, int slot_d,
                       int norm_slot, int iter);
// x += a p (a = sc[slot_c]/sc[slot_d]); p = r + b p (b = sc[slot_cn]/sc[slot_c]); ap = A p.  init: p = r, ap = A p only.
// iter: CG iteration this launch belongs to (systems that converged before it are left untouched)
dwf_status launch_cg_xp(dwf_ctx* c, void* x, void* p, const void* r, void* ap, int prec, int slot_c, int slot_d,
                        int slot_cn, int init, int iter);
dwf_status dhop_time_begin(dwf_ctx* c);
dwf_status dhop_time_end(dwf_ctx* c, double alg_bytes);
dwf_status dhop_timing_flush(dwf_ctx* c);   // synchronises the stream, folds recorded event pairs into dhop_ms

enum { SLOT_C = 0, SLOT_D, SLOT_CN, SLOT_B, SLOT_T0, SLOT_T1, NSLOTS = 16 };
constexpr int CG_RING = 4;

}  // namespace dwf
