/* dwf.h — C-ABI boundary of the B200-native domain-wall-fermion hot path (arXiv:2203.17119).
 *
 * What the library computes (definitions in DESIGN.md §2, readings C1-C10):
 *   - the 4-D Wilson hopping term Dhop over all Ls fifth-dimension slices,
 *   - the 5-D Moebius/Shamir terms (Meooe5D "A", Mooee, Mooee^-1),
 *   - the Dirichlet-cut operator D_Omega (+) D_Omegabar (eqs. 3-4, PAPER.md:175:
 *     "applies Dirichlet boundary conditions to its gauge field argument"),
 *   - the red-black Schur operator Mpc and CG on Mpc^dag Mpc in fp64 and fp32-inner/fp64-outer
 *     ("the usual red-black preconditioned HMC can be used"),
 *   - the full-system red-black solve M psi = eta that the paper's eq. 5 Schur check needs.
 *
 * Conventions
 *   Pointers named *_dev are DEVICE pointers, *_host are HOST pointers.  Field buffers are
 *   owned by the caller (PyTorch allocates them); the context owns its gauge copies, its 5-D
 *   coefficient tables and its solver workspace.  All work is enqueued on the context's CUDA
 *   stream (dwf_set_stream); only dwf_cg / dwf_solve / dwf_norm2 / *_host calls synchronise
 *   that stream, because they return scalars or host data.
 *   A context is single-threaded and single-stream: its calls must not run concurrently with one another (the persistent
 *   Dhop kernels share a tile-queue counter per context, the solver workspace is shared), and after dwf_set_stream the
 *   caller orders the old stream's work before the new one's.  A context belongs to the CUDA device that was current at
 *   dwf_create; every call makes that device current for its duration and restores the caller's afterwards.
 *   Every function returns a dwf_status; nothing throws or aborts across this boundary.
 *   dwf_last_error(ctx) gives a human-readable message for the last failure on ctx.
 *
 * Layouts
 *   CANONICAL (interchange, what the oracle also uses), real type = double or float, C order:
 *     gauge   [lex][mu][row][col][re,im]        lex = ((t*Lz+z)*Ly+y)*Lx+x, mu = 0..3 = x,y,z,t,
 *                                               U_mu(x) is the link from x to x+mu_hat (18 reals)
 *     FULL    [lex][s][spin][colour][re,im]
 *     EVEN/ODD[cb][s][spin][colour][re,im]      cb = lex/2 over sites with (x+y+z+t)%2 == parity
 *   NATIVE (opaque to the caller; dwf_field_bytes gives the size): a tiled, site-vectorised SoA,
 *     16-byte vectors, described in DESIGN.md §4.  A FULL native field is the EVEN native field
 *     followed by the ODD native field.
 */
#ifndef DWF_H
#define DWF_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dwf_ctx dwf_ctx; /* opaque, library-owned */

typedef enum {
    DWF_OK = 0,
    DWF_EINVAL = 1,   /* bad argument: odd dims, Ls < 1 or > 32, cut not dividing, null/aliased pointers */
    DWF_ENOMEM = 2,   /* device allocation failed */
    DWF_ECUDA = 3,    /* a CUDA call or kernel launch failed */
    DWF_ESTATE = 4,   /* gauge field not set */
    DWF_ENOTCONV = 5  /* max_iter reached; x holds the best iterate, info is filled */
} dwf_status;

typedef enum { DWF_F32 = 0, DWF_F64 = 1 } dwf_prec;
typedef enum { DWF_EVEN = 0, DWF_ODD = 1, DWF_FULL = 2 } dwf_parity; /* parity of the OUTPUT field */
typedef enum { DWF_CG_F64 = 0, DWF_CG_MIXED = 1 } dwf_cg_mode;

typedef struct {
    int iters_total;     /* CG iterations, all restarts / inner solves included */
    int iters_inner;     /* fp32 inner iterations (mixed mode), else 0 */
    int restarts;        /* fp64: true-residual restarts; mixed: outer defect-correction steps */
    double resid_iter;   /* recurrence residual |r|/|b| at exit */
    double resid_true;   /* |b - A x|/|b| recomputed at exit (fp64) */
    double resid_full;   /* dwf_solve only: |eta - M psi|/|eta| */
    double seconds;      /* wall time of the call, enqueue to synchronise */
    int launches;        /* kernels launched by the call */
} dwf_cg_info;

/* Create a context for an Lx*Ly*Lz*Lt lattice (all even) with Ls slices (1..32).
 * Moebius parameters: D_+ = b5 D_W + 1, D_- = c5 D_W - 1, D_W = (4-M5) - Dhop/2 (reading C4);
 * Shamir is (b5,c5) = (1,0).  dirichlet_cut[mu] = B > 0 (B divides L_mu) zeroes U_mu(x) for all x
 * with x_mu mod B == B-1 (reading C7); 0 = no cut in that direction.
 * Antiperiodic time boundary by default (reading C2). */
dwf_status dwf_create(dwf_ctx** out, const int dims[4], int Ls, double M5, double mf, double b5, double c5,
                      const int dirichlet_cut[4]);
dwf_status dwf_destroy(dwf_ctx* ctx);

/* Options (set before dwf_set_gauge unless noted):
 *   "antiperiodic_t" 0/1 (default 1)       "compress12" 0/1 (default 1; 2-row links, reading C10)
 *   "tile_x","tile_y","tile_z","tile_t"    native tile extents (default 4, or 2 where 4 does not divide)
 *   "inner_tol" (default 1e-4), "max_restarts" (default 20)     mixed-precision CG (reading C9), any time
 *   "time_dhop" 0/1: bracket every Dhop kernel launch with CUDA events on the context stream (restarts the
 *   accumulators); dwf_get_option "dhop_ms" / "dhop_timed" / "dhop_bytes" then synchronise and return the summed
 *   kernel time, the number of launches timed and their summed algorithmic bytes (bench.py's roofline figure)
 *   "fuse" 0/1 (default 1), any time: Mpc / CG use the Dhop kernel's fused Mee epilogue and the streaming CG column
 *   kernels where the TMA Dhop kernel applies (4^4 tiles, 2-row links); get "fused_active" tells whether they do
 *   "dhop_kernel" 0 auto / 1 shape-generic / 2 cp.async tile kernel and "dhop_dynamic" 0 static round-robin / 1 global
 *   in-order tile queue select among code paths that compute the same result (used by the parity tests), any time.
 *   Unknown keys return DWF_EINVAL. */
dwf_status dwf_set_option(dwf_ctx* ctx, const char* key, double val);
dwf_status dwf_get_option(const dwf_ctx* ctx, const char* key, double* val);
/* cudaStream_t as void* (torch.cuda.current_stream().cuda_stream); NULL = default stream */
dwf_status dwf_set_stream(dwf_ctx* ctx, void* cuda_stream);

/* Copies a canonical fp64 gauge field (device pointer, V4*4*18 doubles) into the context: applies the
 * Dirichlet cut, builds the 8-legs-per-site native copies (forward U_mu(x), backward U_mu(x-mu)^dag) in
 * fp64 and fp32 (round to nearest) for both parities, optionally 2-row compressed.  When a Dirichlet cut is configured
 * the same copies are also kept WITHOUT the cut (used only inside dwf_boundary_op; every other operator sees the cut
 * links).  The native layout is opaque and precision-specific (fp64 and fp32 fields order the sites of a
 * tile differently): move data between precisions with dwf_convert, never by casting a native buffer.
 * With "compress12" = 1 (the default) the third row of every link is rebuilt as conj(row0 x row1), which is the same
 * operator only for SU(3) links: the call first measures max |row2 - conj(row0 x row1)| over all links and returns
 * DWF_EINVAL (message with the measured defect) when it exceeds 1e-10, an absolute bound that fp64 SU(3) links meet and
 * links that went through single precision (defect ~1e-7) do not; reunitarise those, or set "compress12" = 0 to keep all
 * 18 reals.  Also allocates the solver workspace (10 half fields per precision): DWF_ENOMEM if that fails. */
dwf_status dwf_set_gauge(dwf_ctx* ctx, const void* U_dev_canonical_f64);

/* Bytes of a native field of the given precision and parity (DWF_FULL = 2 x half). */
size_t dwf_field_bytes(const dwf_ctx* ctx, dwf_prec prec, dwf_parity parity);
/* canonical (device, same precision) <-> native (device) */
dwf_status dwf_pack(dwf_ctx* ctx, void* native_dev, const void* canonical_dev, dwf_prec prec, dwf_parity parity);
dwf_status dwf_unpack(dwf_ctx* ctx, void* canonical_dev, const void* native_dev, dwf_prec prec, dwf_parity parity);
/* native -> native precision conversion (round to nearest) */
dwf_status dwf_convert(dwf_ctx* ctx, void* dst_dev, dwf_prec dst_prec, const void* src_dev, dwf_prec src_prec,
                       dwf_parity parity);

/* ---- operators: DEVICE pointers to NATIVE fields owned by the caller; out must not alias in ---- */
/* Dhop psi(x,s) = sum_mu [(1-g_mu) U_mu(x) psi(x+mu,s) + (1+g_mu) U_mu(x-mu)^dag psi(x-mu,s)], reading C3;
 * out_parity EVEN/ODD: in is the opposite-parity half field; FULL: both FULL.  dagger swaps the projectors. */
dwf_status dwf_dhop(dwf_ctx* ctx, void* out_dev, const void* in_dev, dwf_parity out_parity, int dagger, dwf_prec prec);
/* site-local 5-D operators (reading C5); parity only selects the field size */
dwf_status dwf_meooe5d(dwf_ctx* ctx, void* out_dev, const void* in_dev, dwf_parity parity, int dagger, dwf_prec prec);
dwf_status dwf_mooee(dwf_ctx* ctx, void* out_dev, const void* in_dev, dwf_parity parity, int dagger, dwf_prec prec);
dwf_status dwf_mooee_inv(dwf_ctx* ctx, void* out_dev, const void* in_dev, dwf_parity parity, int dagger, dwf_prec prec);
/* full unpreconditioned M = Mooee + Meooe on FULL fields (reading C4) */
dwf_status dwf_m(dwf_ctx* ctx, void* out_dev, const void* in_dev, int dagger, dwf_prec prec);
/* Schur operator Mpc = Moo - Moe Mee^-1 Meo on ODD fields (reading C6) */
dwf_status dwf_mpc(dwf_ctx* ctx, void* out_dev, const void* in_dev, int dagger, dwf_prec prec);
/* Mpc^dag Mpc on ODD fields */
dwf_status dwf_mdagm(dwf_ctx* ctx, void* out_dev, const void* in_dev, dwf_prec prec);

/* sum |v|^2 over a native field, accumulated in fp64 with a fixed reduction tree (deterministic) */
dwf_status dwf_norm2(dwf_ctx* ctx, const void* v_dev, dwf_prec prec, dwf_parity parity, double* result_host);

/* The same sum for callers that must not allocate device memory.  dwf_norm2 above, like every solver here, keeps its
 * per-block partial sums in a buffer its context gets from cudaMalloc.  That rules the library out for programs that have
 * handed the whole device to their own memory pool at start-up (lattice codes and tensor frameworks do: a library's
 * cudaMalloc then fails or eats into the pool), for latency-critical paths that cannot take the device-wide synchronisation
 * a cudaMalloc / cudaFree implies, and for plug-ins whose host forbids allocation in its callbacks.  This entry point needs
 * no context and calls no cudaMalloc, cudaFree or allocating library routine: its partial sums go to a fixed 512 KiB array
 * inside the library image (present on every GPU that loads the library, until the process exits).
 *   v_dev       DEVICE pointer, 16-byte aligned, nreal reals of precision prec, any layout (a native or canonical field of
 *               any parity, or any other array); read only.  nreal: a multiple of 2 (fp64) / 4 (fp32); 0 gives 0.0.
 *   result_dev  DEVICE pointer to one double owned by the caller, 8-byte aligned; written by the last kernel enqueued.
 *   cuda_stream cudaStream_t as void* (NULL = default stream).  Two kernels are enqueued, nothing is synchronised: read
 *               *result_dev after ordering against that stream.  The device is the one current at the call.
 *   errbuf      optional HOST buffer of errbuf_len bytes for a message when the status is not DWF_OK (may be NULL).
 * Limit: nreal * sizeof(real) <= DWF_NORM2_STATIC_MAX_BYTES (4 GiB: one partial per 64 KiB of input, 65536 slots).  A larger
 *   input returns DWF_EINVAL and enqueues nothing; so do null / misaligned pointers.  DWF_ECUDA: a runtime call failed.
 * Sharing: all calls on one device use the same array.  Nothing in it has to be zero beforehand (a call writes every slot
 *   it later reads), but calls that may overlap on the GPU - other streams, other threads - race on it: order them.
 * First call on each device: looks up the array's device address once (cudaGetSymbolAddress) and caches it; make that call
 *   outside any stream capture.  Accumulation in fp64 with a fixed tree that depends on nreal only: the same input gives
 *   the same bits on every run and every GPU; it agrees with dwf_norm2 to rounding (a different, also fixed, tree). */
#define DWF_NORM2_STATIC_MAX_BYTES 4294967296ull
dwf_status dwf_norm2_static(const void* v_dev, size_t nreal, dwf_prec prec, double* result_dev, void* cuda_stream,
                            char* errbuf, size_t errbuf_len);

/* CG on Mpc^dag Mpc x = b (reading C8; mixed: C9).  x_dev: in = initial guess (use_guess != 0) else ignored,
 * out = solution; both fp64 native ODD fields.  tol is relative to |b|.  Restarts from the true residual
 * until |b - A x| <= tol |b|.  Returns DWF_ENOTCONV if max_iter is reached: max_iter bounds iters_total, the iterations
 * counted over all restarts / inner solves (for a batch: of the system that needed most).  The stopping test is evaluated on the device
 * and the host enqueues one iteration ahead of the residual it has read: info->launches may include the kernels of one
 * iteration past the last counted one, which leave x untouched (x is exactly the iterate of iteration iters_total). */
dwf_status dwf_cg(dwf_ctx* ctx, void* x_dev, const void* b_dev, double tol, int max_iter, dwf_cg_mode mode,
                  int use_guess, dwf_cg_info* info);
/* ---- Batched ("multi right-hand side") fields and operators ("four PV local solves, and
 * two non-local light quark solves" per force evaluation: the Hasenbusch / Pauli-Villars terms are solves with
 * the same operator on other sources).  N <= 16 systems that share the context's gauge field and parameters are kept in ONE
 * native half field whose fifth dimension is N * Ls long (slice rhs * Ls + s): dwf_mrhs_field_bytes bytes, device memory
 * owned by the caller; dwf_mrhs_insert / dwf_mrhs_extract copy system j from / to an ordinary native half field of the same
 * precision and parity.  The Dhop kernel then loads the 8 links of a site once for N * Ls slices (algorithmic bytes per 5-D
 * site: 48 B + 8 g B / (N Ls), g = 12 or 18 reals, B = 4 or 8), and every other kernel of Mpc / CG runs once for the whole
 * batch.  dwf_cg_mrhs runs N independent CGs (readings C8 / C9 per system: own alpha, beta, stopping test, restarts) that
 * share the launches; a system that has converged is frozen while the others go on.  info: array of nrhs entries.
 * dwf_mrhs_reserve allocates the batched solver workspace (8 batched half fields per precision) ahead of time; otherwise
 * the first batched Mpc / CG call with a larger nrhs does.  Status codes as the single-system calls (dwf_cg_mrhs:
 * DWF_ENOTCONV if any system has not converged at max_iter iterations).  out_parity: DWF_EVEN or DWF_ODD. */
dwf_status dwf_mrhs_reserve(dwf_ctx* ctx, int nrhs);
size_t dwf_mrhs_field_bytes(const dwf_ctx* ctx, int nrhs, dwf_prec prec);
dwf_status dwf_mrhs_insert(dwf_ctx* ctx, void* batched_dev, int nrhs, int j, const void* single_dev, dwf_prec prec);
dwf_status dwf_mrhs_extract(dwf_ctx* ctx, void* single_dev, const void* batched_dev, int nrhs, int j, dwf_prec prec);
dwf_status dwf_dhop_mrhs(dwf_ctx* ctx, void* out_dev, const void* in_dev, int nrhs, dwf_parity out_parity, int dagger,
                         dwf_prec prec);
dwf_status dwf_mpc_mrhs(dwf_ctx* ctx, void* out_dev, const void* in_dev, int nrhs, int dagger, dwf_prec prec);
dwf_status dwf_mdagm_mrhs(dwf_ctx* ctx, void* out_dev, const void* in_dev, int nrhs, dwf_prec prec);
dwf_status dwf_cg_mrhs(dwf_ctx* ctx, void* x_dev, const void* b_dev, int nrhs, double tol, int max_iter, dwf_cg_mode mode,
                       int use_guess, dwf_cg_info* info);

/* Multishift CG (the solver behind rational functions of D^dag D in the DD-RHMC one-flavour action,
 * eqs. 20-21): (Mpc^dag Mpc + shifts[i]) x_i = b for i < nshift with one shared Krylov space, fp64.
 * x_dev: OUT, nshift fp64 native ODD fields back to back (field i at byte offset i * dwf_field_bytes(F64, ODD)), start
 * from zero; b_dev: fp64 native ODD field; shifts_host: nshift <= 16 values, ascending, shifts[0] >= 0 is the base system
 * whose recurrence residual is driven to tol |b|; resid_true_host (may be NULL): |b - (A + shift_i) x_i| / |b| recomputed
 * at exit for every i; info->resid_true is their maximum.  Status as dwf_cg (DWF_ENOTCONV at max_iter). */
dwf_status dwf_multishift_cg(dwf_ctx* ctx, void* x_dev, const void* b_dev, const double* shifts_host, int nshift, double tol,
                             int max_iter, dwf_cg_info* info, double* resid_true_host);
/* Chebyshev polynomial filter (the recursively obtained filter functions of the paper's multigrid
 * set-up, Fig. 4 caption PAPER.md:191 and PAPER.md:197): out = T_order(a) in with a = (2 A - (hi + lo)) / (hi - lo),
 * A = Mpc^dag Mpc, by t_0 = in, t_1 = a in, t_{k+1} = 2 a t_k - t_{k-1}.  Native ODD fields of precision prec, device
 * pointers, out != in; hi > lo; order >= 0.  Enqueued on the context stream (no synchronisation). */
dwf_status dwf_chebyshev(dwf_ctx* ctx, void* out_dev, const void* in_dev, double lo, double hi, int order, dwf_prec prec);
/* Domain decomposition objects of the paper.  They need a Dirichlet cut with an EVEN number of blocks
 * in every cut direction (else DWF_EINVAL); dwf_set_gauge then also keeps the links without the cut.
 * Omega = sites whose block indices floor(x_mu / B_mu), summed over the cut directions, are even (eqs. 1-2).
 * dwf_domain_project: out = P in on FULL native fields (out may alias in), which = 0: P_Omega, 1: P_Omegabar, 2: the
 *   boundary projector P_dbar of eq. 8, found by mask-and-shift: sites of Omega with a cut
 *   link, times (1 +- gamma_mu)/2 for Shamir sites on one cut face, times 1 otherwise (reading in DESIGN.md section 2).
 * dwf_boundary_op: FULL fp64 native fields, out != in.  inverse = 0: R phi = P phi - P D_O^-1 D_d D_Ob^-1 D_dbar phi (eqs. 9-10,
 *   PAPER.md:93-97; two Dirichlet solves); inverse != 0: R^-1 phi = P phi - P D^-1 D_dbar_hat phi (eqs. 13-14, PAPER.md:109-111;
 *   one solve with the uncut operator).  Solves as dwf_solve (tol, max_iter, mode); info->iters_total sums them,
 *   info->resid_full is the worst |eta - M psi|/|eta|.  Synchronises. */
dwf_status dwf_domain_project(dwf_ctx* ctx, void* out_dev, const void* in_dev, int which, dwf_prec prec);
dwf_status dwf_boundary_op(dwf_ctx* ctx, void* out_dev, const void* in_dev, int inverse, double tol, int max_iter,
                           dwf_cg_mode mode, dwf_cg_info* info);
/* M psi = eta on FULL fp64 native fields through the red-black wrap (reading C6):
 * eta' = eta_o - Moe Mee^-1 eta_e; Mpc^dag Mpc psi_o = Mpc^dag eta'; psi_e = Mee^-1 (eta_e - Meo psi_o). */
dwf_status dwf_solve(dwf_ctx* ctx, void* psi_dev, const void* eta_dev, double tol, int max_iter, dwf_cg_mode mode,
                     dwf_cg_info* info);

/* ---- end-to-end entry points with HOST buffers in canonical layout (copies inside the call) ---- */
/* out_host = Dhop in_host; canonical fields of the given precision */
dwf_status dwf_dhop_host(dwf_ctx* ctx, void* out_host, const void* in_host, dwf_parity out_parity, int dagger,
                         dwf_prec prec);
/* out_host = Mpc^dag Mpc in_host; canonical ODD fields */
dwf_status dwf_mdagm_host(dwf_ctx* ctx, void* out_host, const void* in_host, dwf_prec prec);
/* x_host = (Mpc^dag Mpc)^-1 b_host from x = 0; canonical ODD fp64 fields; same stopping rule as dwf_cg */
dwf_status dwf_cg_host(dwf_ctx* ctx, void* x_host, const void* b_host, double tol, int max_iter, dwf_cg_mode mode,
                       dwf_cg_info* info);
/* psi_host = M^-1 eta_host; canonical FULL fp64 fields */
dwf_status dwf_solve_host(dwf_ctx* ctx, void* psi_host, const void* eta_host, double tol, int max_iter,
                          dwf_cg_mode mode, dwf_cg_info* info);

/* kernels launched on this context since creation (for bench.py's gpu_launches) */
long long dwf_launch_count(const dwf_ctx* ctx);
const char* dwf_last_error(const dwf_ctx* ctx);
const char* dwf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DWF_H */
