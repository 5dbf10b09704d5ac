"""GPU parity at BASELINE.json's full size, in the launch configuration bench.py times: configs[3] = c4,
32^4 x Ls=12 Moebius, 2-row compressed links, the seeded eps = 0.7 gauge field and Gaussian source of bench.py.

The oracle finishes one operator application at this size in seconds, so the comparison is element by element on the
WHOLE field (stricter than sampled outputs): Dhop in fp64 and fp32, Mpc, Mpc^dag Mpc, and the first iterations of the
red-black CG (recurrence-residual history, then the oracle recomputes the true residual of the GPU iterate)."""
import numpy as np
import pytest

from paper_2203_17119_b200 import inputs

pytestmark = pytest.mark.gpu


def rel(a, b):
    a = np.asarray(a, dtype=np.complex128).ravel()
    b = np.asarray(b, dtype=np.complex128).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def relmax(a, b):
    """max |a - b| / max |b|: one bad site in 3e8 reals is invisible in a relative L2 norm, not here."""
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    return float(np.abs(a - b).max() / np.abs(b).max())


# elementwise bars beside the L2 bars of north_star: an output is a sum of <= 8 x 12 products of O(1) numbers, so a
# single element may be off by ~50 eps relative to the largest one (tolerances)
MAXTOL = {"f64": 5e-13, "f32": 5e-5}


@pytest.fixture(scope="module")
def c4(oracle_built):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2203_17119_b200 import api
    from oracle.dwf_oracle import Oracle
    cfg = inputs.CONFIGS["c4"]
    U = inputs.make_gauge(cfg)
    g = api.from_config(cfg, device="cuda:0")
    g.set_gauge(U)
    orc = Oracle(cfg.dims, cfg.Ls, cfg.M5, cfg.mf, cfg.b5, cfg.c5, antiperiodic_t=cfg.antiperiodic_t, cut=cfg.cut).set_gauge(U)
    odd = inputs.source_half(cfg.dims, cfg.Ls, cfg.source_seed, parity=1)
    yield dict(api=api, cfg=cfg, g=g, orc=orc, odd=odd, U=U)
    g.close()


def test_c4_runs_the_fast_kernels(c4):
    g = c4["g"]
    assert [int(g.get_option(f"tile_{k}")) for k in "xyzt"] == [4, 4, 4, 4]
    assert g.get_option("compress12") == 1 and g.get_option("fused_active") == 1


def test_c4_dhop_fp64_full_field(c4):
    A, g, orc, odd = c4["api"], c4["g"], c4["orc"], c4["odd"]
    got, want = g.unpack(g.dhop(g.pack(odd, A.F64, A.ODD), A.EVEN, False, A.F64), A.F64, A.EVEN), orc.dhop(odd, 0, False)
    assert rel(got, want) < 1e-12 and relmax(got, want) < MAXTOL["f64"]
    got, want = g.unpack(g.dhop(g.pack(odd, A.F64, A.ODD), A.EVEN, True, A.F64), A.F64, A.EVEN), orc.dhop(odd, 0, True)
    assert rel(got, want) < 1e-12 and relmax(got, want) < MAXTOL["f64"]


def test_c4_dhop_fp32_full_field(c4):
    from oracle.dwf_oracle import Oracle
    A, g, cfg, odd = c4["api"], c4["g"], c4["cfg"], c4["odd"]
    U32 = c4["U"].astype(np.complex64).astype(np.complex128)
    orc32 = Oracle(cfg.dims, cfg.Ls, cfg.M5, cfg.mf, cfg.b5, cfg.c5, antiperiodic_t=cfg.antiperiodic_t, cut=cfg.cut).set_gauge(U32)
    src = odd.astype(np.complex64).astype(np.complex128)
    got, want = g.unpack(g.dhop(g.pack(src, A.F32, A.ODD), A.EVEN, False, A.F32), A.F32, A.EVEN), orc32.dhop(src, 0, False)
    assert rel(got, want) < 1e-5 and relmax(got, want) < MAXTOL["f32"]


def test_c4_mpc_and_mdagm_full_field(c4):
    A, g, orc, odd = c4["api"], c4["g"], c4["orc"], c4["odd"]
    nat = g.pack(odd, A.F64, A.ODD)
    for got, want, f in ((g.unpack(g.mpc(nat, False, A.F64), A.F64, A.ODD), orc.mpc(odd), 1),
                         (g.unpack(g.mpc(nat, True, A.F64), A.F64, A.ODD), orc.mpc(odd, dagger=True), 1),
                         (g.unpack(g.mdagm(nat, A.F64), A.F64, A.ODD), orc.mdagm(odd), 2)):
        assert rel(got, want) < f * 1e-12 and relmax(got, want) < 2 * f * MAXTOL["f64"]


def test_c4_cg_first_iterations_match_oracle(c4):
    """A full oracle CG at this size costs ~10 s per iteration x 254 iterations; reading of SURVEY 8(d): residual-history
    agreement over the first K iterations, then the oracle recomputes the true residual of the GPU iterate."""
    from oracle.dwf_oracle import cg
    A, g, orc, odd = c4["api"], c4["g"], c4["orc"], c4["odd"]
    K = 4
    hist = []
    cg(orc, odd, 1e-30, K, history=hist, restart_on_true=False)
    nat = g.pack(odd, A.F64, A.ODD)
    for k in range(1, K + 1):
        x, info, st = g.cg(nat, 1e-30, k, A.CG_F64)
        assert st == A.ENOTCONV and info["iters_total"] == k
        assert abs(info["resid_iter"] - hist[k - 1]) <= 1e-10 * hist[k - 1], (k, info, hist)
    xs = g.unpack(x, A.F64, A.ODD)
    true_res = np.sqrt(orc.norm2(odd - orc.mdagm(xs)) / orc.norm2(odd))
    assert abs(info["resid_true"] - true_res) <= 1e-9 * true_res


@pytest.mark.parametrize("mode", ["f64", "mixed"])
def test_c4_converged_solution_certified_by_the_oracle(c4, mode):
    """BASELINE configs[3]: "red-black CG to 1e-8 fp64" (and the fp32-inner variant) on the headline lattice, run to
    convergence on the GPU; the oracle then recomputes |b - Mpc^dag Mpc x| / |b| of the returned solution with one
    application of its own operator (SURVEY 8(d) reading (3)): it must meet the tolerance and confirm the residual the
    library reports about itself."""
    A, g, orc, odd, cfg = c4["api"], c4["g"], c4["orc"], c4["odd"], c4["cfg"]
    tol = cfg.tol
    assert tol == 1e-8
    x, info, st = g.cg(g.pack(odd, A.F64, A.ODD), tol, 20000, A.CG_MIXED if mode == "mixed" else A.CG_F64)
    assert st == A.OK and info["resid_true"] <= tol and info["iters_total"] > 100
    if mode == "mixed":
        assert info["iters_inner"] == info["iters_total"] and info["restarts"] >= 1
    xs = g.unpack(x, A.F64, A.ODD)
    del x
    true_res = np.sqrt(orc.norm2(odd - orc.mdagm(xs)) / orc.norm2(odd))
    assert true_res <= tol * (1 + 1e-6), (true_res, info)
    assert abs(true_res - info["resid_true"]) <= 1e-6 * true_res, (true_res, info)


# ---- BASELINE configs[2] = c3: 24^4 x Ls=16 Moebius, eps = 0.5: Dhop in both precisions, mixed-precision CG to 1e-10
@pytest.fixture(scope="module")
def c3(oracle_built):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2203_17119_b200 import api
    from oracle.dwf_oracle import Oracle
    cfg = inputs.CONFIGS["c3"]
    U = inputs.make_gauge(cfg)
    g = api.from_config(cfg, device="cuda:0")
    g.set_gauge(U)
    orc = Oracle(cfg.dims, cfg.Ls, cfg.M5, cfg.mf, cfg.b5, cfg.c5, antiperiodic_t=cfg.antiperiodic_t, cut=cfg.cut).set_gauge(U)
    odd = inputs.source_half(cfg.dims, cfg.Ls, cfg.source_seed, parity=1)
    yield dict(api=api, cfg=cfg, g=g, orc=orc, odd=odd)
    g.close()


def test_c3_dhop_both_precisions_full_field(c3):
    A, g, orc, odd = c3["api"], c3["g"], c3["orc"], c3["odd"]
    got = g.unpack(g.dhop(g.pack(odd, A.F64, A.ODD), A.EVEN, False, A.F64), A.F64, A.EVEN)
    want = orc.dhop(odd, 0, False)
    assert rel(got, want) < 1e-12 and relmax(got, want) < MAXTOL["f64"]
    # fp32 kernel on the fp32-rounded source; its links are the fp64 links rounded to nearest (reading C10), so the
    # fp64 oracle on unrounded links differs by the link rounding too: 1e-5 bar of the north star
    src = odd.astype(np.complex64).astype(np.complex128)
    got32 = g.unpack(g.dhop(g.pack(src, A.F32, A.ODD), A.EVEN, False, A.F32), A.F32, A.EVEN)
    want32 = orc.dhop(src, 0, False)
    assert rel(got32, want32) < 1e-5 and relmax(got32, want32) < MAXTOL["f32"]


def test_c3_mixed_precision_cg_to_1e10(c3):
    A, g, orc, odd, cfg = c3["api"], c3["g"], c3["orc"], c3["odd"], c3["cfg"]
    x, info, st = g.cg(g.pack(odd, A.F64, A.ODD), cfg.tol, 50000, A.CG_MIXED)
    assert st == A.OK and info["resid_true"] <= cfg.tol and 1 <= info["restarts"] <= 20
    xs = g.unpack(x, A.F64, A.ODD)
    true_res = np.sqrt(orc.norm2(odd - orc.mdagm(xs)) / orc.norm2(odd))      # the oracle recomputes it
    assert true_res <= cfg.tol * (1 + 1e-6)
    assert abs(true_res - info["resid_true"]) <= 1e-6 * true_res + 1e-16


def test_c4_results_are_bit_reproducible_and_schedule_independent(c4):
    """every tile is computed by one CTA in a fixed order and the |.|^2 sums are fixed-tree per tile, so the
    operators and the CG scalars must not depend on the run or on the tile scheduling (global queue vs static round-robin)."""
    import torch
    A, g, odd = c4["api"], c4["g"], c4["odd"]
    nat = g.pack(odd, A.F64, A.ODD)
    ref = g.mdagm(nat, A.F64)
    _, info_ref, _ = g.cg(nat, 1e-30, 3, A.CG_F64)
    for dyn in (1, 0, 1):
        g.set_option("dhop_dynamic", dyn)
        assert torch.equal(g.mdagm(nat, A.F64), ref)
        _, info, _ = g.cg(nat, 1e-30, 3, A.CG_F64)
        assert info["resid_iter"] == info_ref["resid_iter"] and info["resid_true"] == info_ref["resid_true"]
    g.set_option("dhop_dynamic", 1)


# ---- BASELINE configs[4] = c5: 32^3 x 64 x Ls=16 Moebius, Haar + 4 APE passes, Dirichlet cut in t into two 32^4 domains
@pytest.fixture(scope="module")
def c5(oracle_built):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2203_17119_b200 import api
    from oracle.dwf_oracle import Oracle
    cfg = inputs.CONFIGS["c5"]
    U = inputs.make_gauge(cfg)
    g = api.from_config(cfg, device="cuda:0")
    g.set_gauge(U)
    orc = Oracle(cfg.dims, cfg.Ls, cfg.M5, cfg.mf, cfg.b5, cfg.c5, antiperiodic_t=cfg.antiperiodic_t, cut=cfg.cut).set_gauge(U)
    odd = inputs.source_half(cfg.dims, cfg.Ls, cfg.source_seed, parity=1)
    yield dict(api=api, cfg=cfg, g=g, orc=orc, odd=odd, U=U)
    g.close()


def test_c5_operators_full_field(c5):
    """Whole-field parity at c5 on the Haar + APE field with the t cut: Dhop fp64 and fp32, Mpc, Mpc^dag Mpc."""
    from oracle.dwf_oracle import Oracle
    A, g, orc, odd, cfg = c5["api"], c5["g"], c5["orc"], c5["odd"], c5["cfg"]
    assert [int(g.get_option(f"tile_{k}")) for k in "xyzt"] == [4, 4, 4, 4] and g.get_option("fused_active") == 1
    nat = g.pack(odd, A.F64, A.ODD)
    got, want = g.unpack(g.dhop(nat, A.EVEN, False, A.F64), A.F64, A.EVEN), orc.dhop(odd, 0, False)
    assert rel(got, want) < 1e-12 and relmax(got, want) < MAXTOL["f64"]
    # fp32 (daggered, for variety) against the fp64 oracle on the fp32-rounded links and source
    U32 = c5["U"].astype(np.complex64).astype(np.complex128)
    orc32 = Oracle(cfg.dims, cfg.Ls, cfg.M5, cfg.mf, cfg.b5, cfg.c5, antiperiodic_t=cfg.antiperiodic_t, cut=cfg.cut).set_gauge(U32)
    src = odd.astype(np.complex64).astype(np.complex128)
    got, want = g.unpack(g.dhop(g.pack(src, A.F32, A.ODD), A.EVEN, True, A.F32), A.F32, A.EVEN), orc32.dhop(src, 0, True)
    assert rel(got, want) < 1e-5 and relmax(got, want) < MAXTOL["f32"]
    del orc32, U32, src
    got, want = g.unpack(g.mpc(nat, False, A.F64), A.F64, A.ODD), orc.mpc(odd)
    assert rel(got, want) < 1e-12 and relmax(got, want) < 2 * MAXTOL["f64"]
    got, want = g.unpack(g.mdagm(nat, A.F64), A.F64, A.ODD), orc.mdagm(odd)
    assert rel(got, want) < 2e-12 and relmax(got, want) < 4 * MAXTOL["f64"]


def test_c5_cg_first_iterations_and_mixed_solution(c5):
    """SURVEY 8(d) reading for sizes where a full oracle CG costs hours: recurrence-residual history over the first K
    iterations, then the oracle recomputes the true residual of the GPU's mixed-precision solution (tol 1e-8, config text)."""
    from oracle.dwf_oracle import cg
    A, g, orc, odd, cfg = c5["api"], c5["g"], c5["orc"], c5["odd"], c5["cfg"]
    K = 3
    hist = []
    cg(orc, odd, 1e-30, K, history=hist, restart_on_true=False)
    nat = g.pack(odd, A.F64, A.ODD)
    for k in range(1, K + 1):
        x, info, st = g.cg(nat, 1e-30, k, A.CG_F64)
        assert st == A.ENOTCONV and info["iters_total"] == k
        assert abs(info["resid_iter"] - hist[k - 1]) <= 1e-10 * hist[k - 1], (k, info, hist)
    x, info, st = g.cg(nat, cfg.tol, 50000, A.CG_MIXED)
    assert st == A.OK and info["resid_true"] <= cfg.tol and 1 <= info["restarts"] <= 20
    xs = g.unpack(x, A.F64, A.ODD)
    true_res = np.sqrt(orc.norm2(odd - orc.mdagm(xs)) / orc.norm2(odd))
    assert true_res <= cfg.tol * (1 + 1e-6)
    assert abs(true_res - info["resid_true"]) <= 1e-6 * true_res + 1e-16


def test_c4_batched_operators_and_cg_equal_the_single_system_path(c4):
    """NEXT-3 at full size, in the launch configuration run_config --extras times: a batch of 3 systems through
    dwf_dhop_mrhs / dwf_mdagm_mrhs equals the single-system kernels bit for bit (system 0 is the source the whole-field
    oracle comparisons above use), and three CG iterations of the batch reproduce the single-system residuals exactly."""
    import torch
    A, g, odd = c4["api"], c4["g"], c4["odd"]
    n = 3
    nat = [g.pack(odd, A.F64, A.ODD)]
    nat.append(nat[0] * 0.25)
    nat.append(g.mdagm(nat[0], A.F64))
    bb = g.mrhs_gather(nat)
    for j, o in enumerate(g.mrhs_scatter(g.dhop_mrhs(bb, n, A.EVEN, False, A.F64), n)):
        assert torch.equal(o, g.dhop(nat[j], A.EVEN, False, A.F64)), j
    for j, o in enumerate(g.mrhs_scatter(g.mdagm_mrhs(bb, n, A.F64), n)):
        assert torch.equal(o, g.mdagm(nat[j], A.F64)), j
    bb32 = g.mrhs_gather([g.convert(v, A.F64, A.F32, A.ODD) for v in nat], A.F32)
    for j, o in enumerate(g.mrhs_scatter(g.mdagm_mrhs(bb32, n, A.F32), n, A.F32)):
        assert torch.equal(o, g.mdagm(g.convert(nat[j], A.F64, A.F32, A.ODD), A.F32)), j
    x, infos, st = g.cg_mrhs(bb, n, 1e-30, 3)
    assert st == A.ENOTCONV
    for j, xs in enumerate(g.mrhs_scatter(x, n)):
        x1, i1, _ = g.cg(nat[j], 1e-30, 3, A.CG_F64)
        assert torch.equal(xs, x1) and infos[j]["resid_iter"] == i1["resid_iter"] and infos[j]["resid_true"] == i1["resid_true"]


def test_c4_mdagm_fp32_full_field(c4):
    """The fp32 Schur operator at full size (the inner operator of the mixed-precision CG, reading C9) against the fp64
    oracle on the fp32-rounded links and source: 1e-5 relative L2 per Dhop (north_star), 2x for Mpc^dag Mpc, and an
    elementwise bar beside it."""
    from oracle.dwf_oracle import Oracle
    A, g, cfg, odd = c4["api"], c4["g"], c4["cfg"], c4["odd"]
    U32 = c4["U"].astype(np.complex64).astype(np.complex128)
    orc32 = Oracle(cfg.dims, cfg.Ls, cfg.M5, cfg.mf, cfg.b5, cfg.c5, antiperiodic_t=cfg.antiperiodic_t, cut=cfg.cut).set_gauge(U32)
    src = odd.astype(np.complex64).astype(np.complex128)
    got, want = g.unpack(g.mdagm(g.pack(src, A.F32, A.ODD), A.F32), A.F32, A.ODD), orc32.mdagm(src)
    assert rel(got, want) < 2e-5 and relmax(got, want) < 4 * MAXTOL["f32"]


def test_c5_adjoint_and_positivity_identities_on_the_gpu(c5):
    """Properties that hold at any size (no oracle needed), at c5 in both precisions: <u, Mpc v> = <Mpc^dag u, v> (the dagger
    kernels are the adjoints of the plain ones, reading C4'), and <v, Mpc^dag Mpc v> = |Mpc v|^2 > 0."""
    import torch
    A, g = c5["api"], c5["g"]
    for P, tol in ((A.F64, 1e-12), (A.F32, 2e-5)):
        u = g.new_native(P, A.ODD).normal_()
        v = g.new_native(P, A.ODD).normal_()
        dot = lambda a, b: complex(torch.dot(a.double(), b.double()).item())       # real dot of the re/im interleaved fields
        # native fields are real arrays of (re, im) pairs in the same order for u and v: Re<u, w> = sum of products
        mv, mdu = g.mpc(v, False, P), g.mpc(u, True, P)
        lhs, rhs = dot(u, mv).real, dot(mdu, v).real
        scale = float(torch.linalg.norm(u.double()) * torch.linalg.norm(mv.double()))
        assert abs(lhs - rhs) <= tol * scale * 10, (P, lhs, rhs)
        av = g.mdagm(v, P)
        q = dot(v, av).real
        n2 = g.norm2(mv, P, A.ODD)
        assert q > 0 and abs(q - n2) <= tol * n2 * 10, (P, q, n2)
