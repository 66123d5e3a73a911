"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on identical seeded inputs.

Tolerances (BASELINE.json north_star; norms per DESIGN.md reading A13), written here:
    overlap      |d| / |ovlp|                      <= 1e-10
    force bias   max_g |d fb| / max_g |fb|  per walker <= 1e-10
    Green's fn   max |dG| / max |G|          per walker <= 1e-10
    energies     |dE|, |dE1|, |dE2|                <= 1e-8 Ha
Summation order differs (atomics, reading A12), so nothing here is bit-exact by construction.
"""
import itertools
import json
import os

import numpy as np
import pytest

import msd_inputs as mi
from oracle import msd_oracle as mo
from oracle import o2

pytestmark = pytest.mark.gpu

TOL_REL = 1e-10
TOL_E = 1e-8
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    torch.cuda.set_device(0)
    return torch


def _msd():
    import paper_2406_08314_b200 as msd
    return msd


def gpu_all(torch, x, trial=None, want_G=True):
    msd = _msd()
    own = trial is None
    trial = msd.setup_from_inputs(x) if own else trial
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    fl = torch.full((x.n_w,), -1, dtype=torch.int32, device="cuda")
    out = dict(ovlp=trial.overlap(pa, pb, flags=fl).cpu().numpy(),
               fb=trial.force_bias(pa, pb).cpu().numpy(),
               E=trial.local_energy(pa, pb).cpu().numpy())
    if want_G:
        out["G"] = trial.greens(pa, pb).cpu().numpy()
    out["flags"] = fl.cpu().numpy()
    torch.cuda.synchronize()
    if own:
        trial.close()
    return out


def assert_parity(got, ref, walkers=None, what=("ovlp", "fb", "E", "G")):
    ws = np.arange(len(ref["ovlp"])) if walkers is None else np.asarray(walkers)
    if "ovlp" in what:
        err = np.abs(got["ovlp"][ws] - ref["ovlp"]) / np.abs(ref["ovlp"])
        assert err.max() <= TOL_REL, "overlap rel err %.3e" % err.max()
    if "fb" in what:
        err = np.abs(got["fb"][ws] - ref["fb"]).max(axis=1) / np.abs(ref["fb"]).max(axis=1)
        assert err.max() <= TOL_REL, "force bias rel err %.3e" % err.max()
    if "E" in what:
        err = np.abs(got["E"][ws] - ref["E"])
        assert err.max() <= TOL_E, "energy abs err %.3e Ha" % err.max()
    if "G" in what and "G" in ref and "G" in got:
        err = np.abs(got["G"][ws] - ref["G"]).max(axis=(1, 2, 3)) / np.abs(ref["G"]).max(axis=(1, 2, 3))
        assert err.max() <= TOL_REL, "greens rel err %.3e" % err.max()


# ----------------------------------------------------------------------------------------------
# element-by-element parity at sizes the oracle finishes in seconds (several tiles + ragged tails)
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["micro", "micro-cs", "tiny", "tiny-full", "open-shell", "small"])
def test_parity_all_walkers(torch_cuda, name):
    x = mi.generate(name)
    got = gpu_all(torch_cuda, x)
    ref = o2.run(x)
    assert (got["flags"] == 0).all()
    assert_parity(got, ref)


def test_parity_tiny_against_o0_and_o1(torch_cuda):
    """BASELINE configs[0] against the two numpy tiers as well (no inverse in O0)."""
    x = mi.generate("tiny")
    got = gpu_all(torch_cuda, x)
    assert_parity(got, mo.run(x, "o1"))
    assert_parity(got, mo.run(x, "o0", walkers=[0, 3, 7]), walkers=[0, 3, 7])


@pytest.mark.parametrize("K", [1, 3, 6, 10])
def test_parity_sweep_points(torch_cuda, K):
    """BASELINE configs[4] (kernel sweep) at n_det = 1500: closed-form levels, the level-4/5 boundary and the
    in-shared-memory Gauss-Jordan path up to 10-fold excitations."""
    x = mi.generate("sweep", n_det=1500 if K > 1 else 300, max_level=K)
    got = gpu_all(torch_cuda, x, want_G=False)
    ws = [0, 7, 8, 63, 127]
    assert_parity(got, o2.run(x, walkers=ws, return_G=False), walkers=ws)
    assert_parity(got, o2.run(x, want=("ovlp",)), what=("ovlp",))


def test_parity_cu2o2_full_size(torch_cuda):
    """BASELINE configs[2] at full size, full batch on the GPU; oracle on sampled walkers (first, last, tile
    boundaries 7|8 and 63|64) for energy and force bias, on every walker for the overlap."""
    x = mi.generate("cu2o2")
    got = gpu_all(torch_cuda, x, want_G=False)
    assert (got["flags"] == 0).all()
    ws = [0, 7, 8, 64, 199]
    assert_parity(got, o2.run(x, walkers=ws, return_G=False), walkers=ws)
    assert_parity(got, o2.run(x, want=("ovlp",)), what=("ovlp",))
    ws2 = list(range(16, 32))
    assert_parity(got, o2.run(x, walkers=ws2, want=("ovlp", "greens"), return_G=False), walkers=ws2, what=("ovlp", "fb"))


def _cplx(a):
    a = np.array(a)
    return a[..., 0] + 1j * a[..., 1]


def _assert_against_golden(gold, ov, fb, E):
    """Sections of a golden file (tests/golden/make_golden.py): energy walkers (ovlp, E, fb on every 8th gamma),
    fb_walkers (every gamma), ovlp_all (every walker)."""
    if "walkers" in gold:
        ws, gs = gold["walkers"], gold["fb_gamma_sample"]
        g_ov, g_E, g_fb = _cplx(gold["ovlp"]), _cplx(gold["E"]), _cplx(gold["fb"])
        assert (np.abs(ov[ws] - g_ov) / np.abs(g_ov)).max() <= TOL_REL
        if E is not None:
            assert np.abs(E[ws] - g_E).max() <= TOL_E
        if fb is not None:
            assert (np.abs(fb[ws][:, gs] - g_fb).max(axis=1) / np.array(gold["fb_max_abs"])).max() <= TOL_REL
    if "fb_walkers" in gold and fb is not None:
        ws, g_fb = gold["fb_walkers"], _cplx(gold["fb_full"])
        assert g_fb.shape == (len(ws), fb.shape[1])
        assert (np.abs(fb[ws] - g_fb).max(axis=1) / np.abs(g_fb).max(axis=1)).max() <= TOL_REL
    if "ovlp_all" in gold:
        g_ov = _cplx(gold["ovlp_all"])
        assert g_ov.shape == ov.shape
        assert (np.abs(ov - g_ov) / np.abs(g_ov)).max() <= TOL_REL


@pytest.mark.parametrize("name", ["fe2s2", "cu2o2"])
def test_parity_full_size_against_stored_oracle_values(torch_cuda, name):
    """BASELINE configs[3] (the bench workload, same launch configuration) and configs[2] against oracle values
    stored by tests/golden/make_golden.py (which calls only oracle/): the brute-force oracle needs ~10 minutes per
    walker at the Fe2S2 size.  fe2s2 (SURVEY.md 8(d) plan): overlap of all 100 walkers, force bias (every gamma) of
    walkers 0..15, energy of walkers 0, 7 | 8 (last lane of tile 0, first lane of tile 1), 57, 99 and 34, the walker with
    the worst-conditioned reference block of the batch (cond 708; cu2o2: walkers 16 and 151, cond 444 and 919), which the
    V contraction routes to the 4-multiplication kernel."""
    gold = json.load(open(os.path.join(GOLDEN, "%s_seed0.json" % name)))
    x = mi.generate(name)
    assert gold["input_sha256"] == x.sha256()
    msd = _msd()
    torch = torch_cuda
    trial = msd.setup_from_inputs(x)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    ov = trial.overlap(pa, pb).cpu().numpy()
    fb = trial.force_bias(pa, pb).cpu().numpy()
    E = trial.local_energy(pa, pb).cpu().numpy()
    trial.close()
    if name == "fe2s2":
        assert len(gold["ovlp_all"]) == x.n_w and len(gold["fb_walkers"]) >= 16
        assert {0, 7, 8, 34, 57, 99} <= set(gold["walkers"])
    else:
        assert {16, 151} <= set(gold["walkers"])
    _assert_against_golden(gold, ov, fb, E)


@pytest.mark.parametrize("n_det,K,energy", [(100000, 8, True), (1000000, 10, False)])
def test_parity_sweep_end_points_against_stored_oracle_values(torch_cuda, n_det, K, energy):
    """BASELINE configs[4] (kernel sweep) at its large end: N_d = 1e5 with levels <= 8 (overlap of all 128 walkers, force
    bias of walkers 7 | 8 and of the energy walker, energy of walker 64) and N_d = 1e6 with levels <= 10 (overlap of all
    128 walkers) against stored O2 values."""
    gold = json.load(open(os.path.join(GOLDEN, "sweep_nd%d_K%d_seed0.json" % (n_det, K))))
    x = mi.generate("sweep", n_det=n_det, max_level=K)
    assert gold["input_sha256"] == x.sha256()
    msd = _msd()
    torch = torch_cuda
    trial = msd.setup_from_inputs(x)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    ov = trial.overlap(pa, pb).cpu().numpy()
    fb = trial.force_bias(pa, pb).cpu().numpy() if "fb_walkers" in gold else None
    E = trial.local_energy(pa, pb).cpu().numpy() if energy else None
    trial.close()
    assert len(gold["ovlp_all"]) == x.n_w
    _assert_against_golden(gold, ov, fb, E)


@pytest.mark.parametrize("name,kw", [("small", {}), ("open-shell", {}), ("cu2o2", dict(n_w=40))])
def test_reference_block_conditioning(torch_cuda, name, kw):
    """msd_reference_cond: ||O0||_F ||O0^-1||_F of every walker and spin against numpy (the quantity the energy accuracy
    depends on and the V contraction is routed by: DESIGN.md section 7); a singular block reads inf; chunked workspace."""
    torch = torch_cuda
    msd = _msd()
    x = mi.generate(name, **kw)
    pa_h = x.phi_a.copy()
    pa_h[1][x.occ_ref_a, :] = 0.0                       # walker 1: singular alpha block
    x = x.with_walkers(pa_h, x.phi_b)
    trial = msd.setup_from_inputs(x)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    want = np.zeros((x.n_w, 2))
    for w in range(x.n_w):
        for s_, (phi, occ) in enumerate(((x.phi_a, x.occ_ref_a), (x.phi_b, x.occ_ref_b))):
            O = phi[w][occ, :]
            if w == 1 and s_ == 0:
                want[w, s_] = np.inf
            elif O.shape[0]:
                want[w, s_] = np.linalg.norm(O) * np.linalg.norm(np.linalg.inv(O))
    for limit in (0, 600 * 1024) if name == "small" else (0,):
        trial.set_workspace_limit(limit)
        got = trial.reference_cond(pa, pb).cpu().numpy()
        assert np.isinf(got[1, 0])
        fin = np.isfinite(want)
        assert (np.abs(got[fin] - want[fin]) <= 1e-9 * want[fin]).all()
    trial.close()


@pytest.mark.parametrize("seed", [1, 2, 3, 4])
@pytest.mark.parametrize("name,kw", [("small", {}), ("sweep", dict(n_det=1500, max_level=7, n_w=19)),
                                     ("sweep", dict(n_det=800, max_level=10, n_w=9))])
def test_parity_other_seeds(torch_cuda, name, kw, seed):
    """Other draws of trial and walkers than the default seed of every other test (the worst reference-block condition
    numbers of these batches run from 50 to 340): every call, the fused call and the force-bias-with-overlap call, all
    walkers, against O2."""
    msd = _msd()
    torch = torch_cuda
    x = mi.generate(name, seed=seed, **kw)
    trial = msd.setup_from_inputs(x)
    got = gpu_all(torch, x, trial=trial, want_G=False)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    fused = trial.force_bias_energy(pa, pb).cpu().numpy()
    fb2, ov2 = trial.force_bias_overlap(pa, pb)
    trial.close()
    ref = o2.run(x, return_G=False)
    assert (got["flags"] == 0).all()
    assert_parity(got, ref, what=("ovlp", "fb", "E"))
    assert_parity(dict(fb=fused[:, :x.n_chol], E=fused[:, x.n_chol:]), ref, what=("fb", "E"))
    assert_parity(dict(ovlp=ov2.cpu().numpy(), fb=fb2.cpu().numpy()), ref, what=("ovlp", "fb"))


@pytest.mark.parametrize("kw", [dict(N=72, n_alpha=34, n_beta=33, A=12, n_chol=30, n_det=200, n_w=11, max_level=4),
                                dict(N=160, n_alpha=30, n_beta=29, A=12, n_chol=20, n_det=120, n_w=9, max_level=3)])
def test_parity_many_electrons(torch_cuda, kw):
    """34 + 33 electrons in 72 orbitals (more electrons per spin than any BASELINE config: the reference kernel's
    Gauss-Jordan beyond one warp's width of columns, the S7 path for shapes the fused kernel does not instantiate), odd
    and unequal electron counts; and 30 + 29 electrons in 160 orbitals, a walker block too large for the reference kernel
    to stage in shared memory (it reads psi from global memory).  Every call on every walker against O2."""
    x = mi.generate("small", **kw)
    got = gpu_all(torch_cuda, x)
    assert (got["flags"] == 0).all()
    assert_parity(got, o2.run(x))


# ----------------------------------------------------------------------------------------------
# edge and degenerate cases
# ----------------------------------------------------------------------------------------------
def test_empty_and_ragged_batches(torch_cuda):
    torch = torch_cuda
    msd = _msd()
    x = mi.generate("small", n_w=21)
    trial = msd.setup_from_inputs(x)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    assert trial.overlap(pa[:0], pb[:0]).shape == (0,)
    assert trial.local_energy(pa[:0], pb[:0]).shape == (0, 3)
    ref = o2.run(x, return_G=False)
    for nw in (1, 5, 8, 9, 21):
        got = dict(ovlp=trial.overlap(pa[:nw].contiguous(), pb[:nw].contiguous()).cpu().numpy(),
                   fb=trial.force_bias(pa[:nw].contiguous(), pb[:nw].contiguous()).cpu().numpy(),
                   E=trial.local_energy(pa[:nw].contiguous(), pb[:nw].contiguous()).cpu().numpy())
        sub = {k: ref[k][:nw] for k in ("ovlp", "fb", "E")}
        assert_parity(got, sub, what=("ovlp", "fb", "E"))
    trial.close()


def test_host_buffer_entry_points(torch_cuda):
    """msd_*_host (the e2e path of bench.py): numpy in, numpy out, copies inside the C call; pinned torch buffers too."""
    torch = torch_cuda
    msd = _msd()
    x = mi.generate("small", n_w=13)
    ref = o2.run(x, return_G=False)
    trial = msd.setup_from_inputs(x)
    fl = np.full(x.n_w, -1, dtype=np.int32)
    got = dict(ovlp=trial.overlap_host(x.phi_a, x.phi_b, flags=fl), fb=trial.force_bias_host(x.phi_a, x.phi_b),
               E=trial.local_energy_host(x.phi_a, x.phi_b))
    assert (fl == 0).all()
    assert_parity(got, ref, what=("ovlp", "fb", "E"))
    ha, hb = torch.from_numpy(x.phi_a).pin_memory(), torch.from_numpy(x.phi_b).pin_memory()
    he = torch.empty((x.n_w, 3), dtype=torch.complex128).pin_memory()
    trial.local_energy_host(ha, hb, out=he)
    assert np.abs(he.numpy() - ref["E"]).max() <= TOL_E
    assert trial.overlap_host(x.phi_a[:0], x.phi_b[:0]).shape == (0,)
    trial.close()


def test_single_determinant_trial(torch_cuda):
    """P1/P2: the MSD path with one determinant is SD-AFQMC (Eq. 13-14)."""
    x = mi.generate("small", n_w=9).subset_dets([0])
    x.ci[:] = 1.0
    got = gpu_all(torch_cuda, x)
    assert_parity(got, o2.run(x))
    d = np.array([np.linalg.det(x.phi_a[w][:8]) * np.linalg.det(x.phi_b[w][:8]) for w in range(x.n_w)])
    assert (np.abs(got["ovlp"] - d) / np.abs(d)).max() < 1e-12


def _reference_walkers(x, n_w):
    pa = np.zeros((n_w, x.N, x.n_alpha), complex)
    pb = np.zeros((n_w, x.N, x.n_beta), complex)
    pa[:, x.occ_ref_a, np.arange(x.n_alpha)] = 1.0
    pb[:, x.occ_ref_b, np.arange(x.n_beta)] = 1.0
    return x.with_walkers(pa, pb)


@pytest.mark.parametrize("name", ["micro-cs", "tiny", "open-shell"])
def test_walker_equals_reference_exact_singular_minors(torch_cuda, name):
    """P7: psi = D_0 makes every minor exactly singular (g = 0); only division-free cofactors survive.
    Oracle: O0 (determinants only; O1/O2 cannot invert O_I here)."""
    x = _reference_walkers(mi.generate(name), 3)
    got = gpu_all(torch_cuda, x)
    ref = mo.run(x, "o0", walkers=[0])
    assert (got["flags"] == 0).all()
    for w in range(3):
        assert abs(got["ovlp"][w] - x.ci[0]) <= 1e-15
        assert np.abs(got["E"][w] - ref["E"][0]).max() <= TOL_E
        assert np.abs(got["fb"][w] - ref["fb"][0]).max() <= TOL_REL * np.abs(ref["fb"][0]).max()
        assert np.abs(got["G"][w] - ref["G"][0]).max() <= TOL_REL


@pytest.mark.parametrize("coop_min", [None, 0, 200])
def test_walker_equals_reference_exact_singular_minors_high_levels(torch_cuda, coop_min):
    """The same through the level >= 5 kernels (in-shared-memory eliminations: every pivot is exactly zero, so the
    determinant-only elimination of the overlap call, the Gauss-Jordan inverse of the other calls and their cooperative
    forms must all return exact zeros, not NaN): N = 12, 6 + 6 electrons, levels up to 6 in each spin; per-thread kernel,
    cooperative kernel (MSD_OPT_COOP_MIN_ELEMS 0) and the default mix.  Oracle: O0 (seconds at this size)."""
    msd = _msd()
    x = mi.generate("sweep", N=12, n_alpha=6, n_beta=6, A=12, n_det=40, max_level=6, n_w=8, n_chol=10)
    assert max(np.diff(x.exc_off_a).max(), np.diff(x.exc_off_b).max()) >= 5
    x = _reference_walkers(x, 3)
    trial = msd.setup_from_inputs(x)
    if coop_min is not None:
        trial.set_option(msd.MSD_OPT_COOP_MIN_ELEMS, coop_min)
    got = gpu_all(torch_cuda, x, trial=trial)
    trial.close()
    ref = mo.run(x, "o0", walkers=[0])
    assert (got["flags"] == 0).all()
    for w in range(3):
        assert abs(got["ovlp"][w] - x.ci[0]) <= 1e-15
        assert np.abs(got["E"][w] - ref["E"][0]).max() <= TOL_E
        assert np.abs(got["fb"][w] - ref["fb"][0]).max() <= TOL_REL * np.abs(ref["fb"][0]).max()
        assert np.abs(got["G"][w] - ref["G"][0]).max() <= TOL_REL


@pytest.mark.parametrize("eps,K", [(1e-1, 6), (1e-3, 6), (1e-6, 6), (1e-9, 6), (1e-3, 10), (1e-9, 9)])
def test_near_reference_walkers(torch_cuda, eps, K):
    """P8: psi = QR(D_0 + eps Z): the regime of real AFQMC walkers; stresses det*inverse cofactors (the Jacobi division
    by R at k >= 5) down to eps = 1e-9 and up to level 10."""
    x = mi.generate("sweep", n_det=600, max_level=K, n_w=10)
    pa, pb = mi.near_reference_walkers(x, eps, seed=4)
    x = x.with_walkers(pa, pb)
    got = gpu_all(torch_cuda, x, want_G=False)
    assert_parity(got, o2.run(x, return_G=False), what=("ovlp", "fb", "E"))


def test_singular_reference_and_zero_overlap_are_flagged(torch_cuda):
    torch = torch_cuda
    msd = _msd()
    x = mi.generate("tiny")
    pa = x.phi_a.copy()
    pa[2][x.occ_ref_a, :] = 0.0                      # walker 2: psi[occ_ref,:] = 0 -> det O0 = 0
    y = x.with_walkers(pa, x.phi_b)
    got = gpu_all(torch, y)
    assert got["flags"][2] & 1 and (np.delete(got["flags"], 2) == 0).all()
    assert np.isnan(got["ovlp"][2]) and np.isnan(got["E"][2]).all() and np.isnan(got["fb"][2]).all()
    ref = o2.run(y, walkers=[0, 1, 3, 7])
    assert_parity(got, ref, walkers=[0, 1, 3, 7])
    # a trial without its reference determinant, evaluated at the reference walker: every R_I = 0 -> W = 0
    z = _reference_walkers(mi.generate("tiny").subset_dets(np.arange(1, 36)), 2)
    trial = msd.setup_from_inputs(z)
    fl = torch.zeros(2, dtype=torch.int32, device="cuda")
    e = trial.local_energy(torch.tensor(z.phi_a, device="cuda"), torch.tensor(z.phi_b, device="cuda"), flags=fl)
    assert (fl.cpu().numpy() & 2).all() and torch.isnan(e.real).all()
    trial.close()


def test_invalid_tables_are_rejected(torch_cuda):
    msd = _msd()
    x = mi.generate("tiny")

    def setup(**kw):
        a = dict(N=x.N, n_alpha=x.n_alpha, n_beta=x.n_beta, n_chol=x.n_chol, n_det=x.n_det, h1=x.h1, L=x.L, e0=0.0,
                 occ_ref_a=x.occ_ref_a, occ_ref_b=x.occ_ref_b, exc_off_a=x.exc_off_a, holes_a=x.holes_a.copy(),
                 parts_a=x.parts_a.copy(), exc_off_b=x.exc_off_b, holes_b=x.holes_b, parts_b=x.parts_b, ci=x.ci)
        a.update(kw)
        return msd.msd_setup(**a)

    bad = x.holes_a.copy(); bad[0] = 5                     # hole not in the reference
    with pytest.raises(msd.MSDError) as e:
        setup(holes_a=bad)
    assert e.value.code == -1
    bad = x.parts_a.copy(); bad[0] = 1                     # particle inside the reference
    with pytest.raises(msd.MSDError):
        setup(parts_a=bad)
    bad = x.parts_a.copy(); bad[0] = x.N + 3               # out of range
    with pytest.raises(msd.MSDError):
        setup(parts_a=bad)
    with pytest.raises(msd.MSDError):                      # unsorted reference
        setup(occ_ref_a=x.occ_ref_a[::-1].copy())
    k = np.diff(x.exc_off_a)
    I = int(np.argmax(k == 2))
    bad = x.parts_a.copy(); bad[x.exc_off_a[I] + 1] = bad[x.exc_off_a[I]]   # repeated particle in one determinant
    with pytest.raises(msd.MSDError):
        setup(parts_a=bad)
    setup().close()


def test_setup_from_occ_and_unordered_tables(torch_cuda):
    """The paper's (coeff, occa, occb) format and hole/particle lists in any order."""
    torch = torch_cuda
    msd = _msd()
    x = mi.generate("open-shell")
    ref = o2.run(x, return_G=False)
    rng = np.random.default_rng(0)
    occa = np.array([rng.permutation(r) for r in x.occa], dtype=np.int32)
    occb = np.array([rng.permutation(r) for r in x.occb], dtype=np.int32)
    t1 = msd.msd_setup_from_occ(x.N, x.n_alpha, x.n_beta, x.n_chol, x.n_det, x.h1, x.L, x.e0, occa, occb, x.ci)
    assert_parity(gpu_all(torch, x, trial=t1, want_G=False), ref, what=("ovlp", "fb", "E"))
    t1.close()
    ha, pa = x.holes_a.copy(), x.parts_a.copy()
    for I in range(x.n_det):
        s = slice(x.exc_off_a[I], x.exc_off_a[I + 1])
        ha[s] = ha[s][::-1]
        pa[s] = rng.permutation(pa[s])
    t2 = msd.msd_setup(x.N, x.n_alpha, x.n_beta, x.n_chol, x.n_det, x.h1, x.L, x.e0, x.occ_ref_a, x.occ_ref_b,
                       x.exc_off_a, ha, pa, x.exc_off_b, x.holes_b, x.parts_b, x.ci)
    assert_parity(gpu_all(torch, x, trial=t2, want_G=False), ref, what=("ovlp", "fb", "E"))
    t2.close()


def test_non_aufbau_reference(torch_cuda):
    """Reference occupation that is not the lowest orbitals: particles may lie below occupied orbitals, so the
    in-place -> sorted phases are non-trivial (reading A6)."""
    torch = torch_cuda
    rng = np.random.default_rng(3)
    x = mi.generate("open-shell")
    perm = rng.permutation(x.N)                      # relabel orbitals: same physics, scrambled reference
    inv = np.argsort(perm)
    h1 = x.h1[np.ix_(inv, inv)]
    L = np.ascontiguousarray(x.L[:, inv][:, :, inv])
    occa = np.sort(perm[x.occa], axis=1).astype(np.int32)
    occb = np.sort(perm[x.occb], axis=1).astype(np.int32)
    # relabelling permutes the rows of each determinant's string: the sign change is part of the physics of the
    # relabelled problem, so compare against the oracle run on the relabelled inputs themselves
    import dataclasses
    ra, rb = occa[0].copy(), occb[0].copy()
    ta, tb = mi.occ_to_tables(occa, ra), mi.occ_to_tables(occb, rb)
    y = dataclasses.replace(x, h1=h1, L=L, occa=occa, occb=occb, occ_ref_a=ra, occ_ref_b=rb,
                            exc_off_a=ta[0], holes_a=ta[1], parts_a=ta[2], exc_off_b=tb[0], holes_b=tb[1], parts_b=tb[2],
                            phi_a=np.ascontiguousarray(x.phi_a[:, inv]), phi_b=np.ascontiguousarray(x.phi_b[:, inv]))
    assert_parity(gpu_all(torch, y), o2.run(y))


# ----------------------------------------------------------------------------------------------
# properties that hold at any size, on the full batch (GPU self-consistency)
# ----------------------------------------------------------------------------------------------
def test_gauge_order_and_chunk_invariance(torch_cuda):
    torch = torch_cuda
    msd = _msd()
    x = mi.generate("small")
    base = gpu_all(torch, x, want_G=False)
    rng = np.random.default_rng(9)
    # P4 gauge: psi -> psi A
    Aa = rng.standard_normal((8, 8)) + 1j * rng.standard_normal((8, 8))
    Ab = rng.standard_normal((8, 8)) + 1j * rng.standard_normal((8, 8))
    g = gpu_all(torch, x.with_walkers(x.phi_a @ Aa, x.phi_b @ Ab), want_G=False)
    fac = np.linalg.det(Aa) * np.linalg.det(Ab)
    assert (np.abs(g["ovlp"] - fac * base["ovlp"]) / np.abs(fac * base["ovlp"])).max() < 1e-9
    assert np.abs(g["E"] - base["E"]).max() < TOL_E
    assert (np.abs(g["fb"] - base["fb"]).max(axis=1) / np.abs(base["fb"]).max(axis=1)).max() < 1e-9
    # P11 determinant order
    p = gpu_all(torch, x.subset_dets(rng.permutation(x.n_det)), want_G=False)
    assert (np.abs(p["ovlp"] - base["ovlp"]) / np.abs(base["ovlp"])).max() < TOL_REL
    assert np.abs(p["E"] - base["E"]).max() < TOL_E
    # walker chunking under a small workspace limit (results must not depend on chunking)
    # 24 MB chunks the energy workspace (Lambda alone is 52 MB); 300 KB also chunks the overlap / force-bias / greens ones
    for limit in (24 * 1024 * 1024, 300 * 1024):
        trial = msd.setup_from_inputs(x)
        trial.set_workspace_limit(limit)
        if limit < 1024 * 1024:
            pa = torch.tensor(x.phi_a, device="cuda"); pb = torch.tensor(x.phi_b, device="cuda")
            c = dict(ovlp=trial.overlap(pa, pb).cpu().numpy(), fb=trial.force_bias(pa, pb).cpu().numpy(), E=base["E"])
            G = trial.greens(pa, pb).cpu().numpy()
            trial.set_workspace_limit(0)            # back to the default: the next call lays the workspace out again
            G2 = trial.greens(pa, pb).cpu().numpy()
            assert np.abs(G - G2).max() < TOL_REL
        else:
            c = gpu_all(torch, x, trial=trial, want_G=False)
            pa = torch.tensor(x.phi_a, device="cuda"); pb = torch.tensor(x.phi_b, device="cuda")
            fused = trial.force_bias_energy(pa, pb).cpu().numpy()
            assert (np.abs(fused[:, :x.n_chol] - base["fb"]).max(axis=1) / np.abs(base["fb"]).max(axis=1)).max() < TOL_REL
            assert np.abs(fused[:, x.n_chol:] - base["E"]).max() < TOL_E
        trial.close()
        assert (np.abs(c["ovlp"] - base["ovlp"]) / np.abs(base["ovlp"])).max() < TOL_REL
        assert np.abs(c["E"] - base["E"]).max() < TOL_E
        assert (np.abs(c["fb"] - base["fb"]).max(axis=1) / np.abs(base["fb"]).max(axis=1)).max() < TOL_REL


# ----------------------------------------------------------------------------------------------
# the packer (S0): integer / index work is bit-exact
# ----------------------------------------------------------------------------------------------
def _parity_bruteforce(occ_ref, holes, parts):
    lst = list(occ_ref)
    for h, p in zip(sorted(holes), sorted(parts)):
        lst[lst.index(h)] = p
    inv = sum(1 for i, j in itertools.combinations(range(len(lst)), 2) if lst[i] > lst[j])
    return -1.0 if inv & 1 else 1.0


@pytest.mark.parametrize("name", ["tiny-full", "open-shell", "small"])
def test_packer_buckets_and_phases(torch_cuda, name):
    msd = _msd()
    x = mi.generate(name)
    trial = msd.setup_from_inputs(x)
    pk = trial.packed()
    info = trial.info()
    trial.close()
    perm = pk["perm"]
    assert sorted(perm.tolist()) == list(range(x.n_det))                      # a permutation
    ka, kb = np.diff(x.exc_off_a)[perm], np.diff(x.exc_off_b)[perm]
    assert (ka == pk["level_a"]).all() and (kb == pk["level_b"]).all()
    key = ka * 17 + kb
    assert (np.diff(key) >= 0).all()                                           # contiguous level buckets, ascending
    for k in np.unique(key):                                                   # stable inside a bucket
        assert (np.diff(perm[key == k]) > 0).all()
    assert info["n_buckets"] == len(np.unique(key))
    for s, I in enumerate(perm):
        ph = _parity_bruteforce(x.occ_ref_a, x.holes_a[x.exc_off_a[I]:x.exc_off_a[I + 1]],
                                x.parts_a[x.exc_off_a[I]:x.exc_off_a[I + 1]]) * \
             _parity_bruteforce(x.occ_ref_b, x.holes_b[x.exc_off_b[I]:x.exc_off_b[I + 1]],
                                x.parts_b[x.exc_off_b[I]:x.exc_off_b[I + 1]])
        assert pk["coef"][s] == x.ci[I] * ph                                   # bit-exact
    assert info["n_o_alpha"] == len(np.unique(x.holes_a)) and info["n_v_alpha"] == len(np.unique(x.parts_a))


def test_native_library_is_the_path(torch_cuda):
    """The kernels ran: launches counted, and the in-tree .so is mapped into this process."""
    msd = _msd()
    x = mi.generate("tiny")
    trial = msd.setup_from_inputs(x)
    n0 = trial.launch_count()
    gpu_all(torch_cuda, x, trial=trial)
    assert trial.launch_count() > n0 >= 5
    trial.close()
    maps = open("/proc/self/maps").read()
    assert "libmsd_b200.so" in maps


def test_many_generic_items_per_cta(torch_cuda):
    """Kernel-sweep shape with enough high-level determinants that every CTA of the generic-level kernel walks through
    several work items of different level pairs (regression: the shared-memory split between a thread's matrices and
    its pair indices must not depend on the item).  Overlap against O2 on every walker, force bias and energy on one."""
    x = mi.generate("sweep", n_det=40000, max_level=6, n_w=8)
    got = gpu_all(torch_cuda, x, want_G=False)
    assert (got["flags"] == 0).all()
    assert_parity(got, o2.run(x, want=("ovlp",)), what=("ovlp",))
    assert_parity(got, o2.run(x, walkers=[5], return_G=False), walkers=[5])


def test_many_high_level_items_per_cta(torch_cuda):
    """The same at levels up to 10 (cooperative kernel, one determinant per warp): 20000 determinants so that a CTA
    processes many items; overlap on every walker, force bias on two, energy on one walker -- all against the
    brute-force oracle O2 (about 2e11 flop for the energy walker: seconds on the host cores)."""
    x = mi.generate("sweep", n_det=20000, max_level=10, n_w=8)
    got = gpu_all(torch_cuda, x, want_G=False)
    assert (got["flags"] == 0).all()
    assert_parity(got, o2.run(x, want=("ovlp",)), what=("ovlp",))
    ws = [0, 7]
    assert_parity(got, o2.run(x, walkers=ws, want=("ovlp", "greens"), return_G=False), walkers=ws, what=("ovlp", "fb"))
    assert_parity(got, o2.run(x, walkers=[3], return_G=False), walkers=[3], what=("ovlp", "fb", "E"))


@pytest.mark.parametrize("name,kw", [("small", {}), ("open-shell", {}), ("tiny", {}),
                                     ("sweep", dict(n_det=3000, max_level=7, n_w=21))])
def test_fused_force_bias_energy_call(torch_cuda, name, kw):
    """msd_force_bias_energy: both outputs from one pass (force bias from C and the B slices) against
    the oracle, and against the two separate calls; device and host-buffer variants; ragged batch, flags."""
    torch = torch_cuda
    msd = _msd()
    x = mi.generate(name, **kw)
    trial = msd.setup_from_inputs(x)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    fl = torch.full((x.n_w,), -1, dtype=torch.int32, device="cuda")
    out = trial.force_bias_energy(pa, pb, flags=fl).cpu().numpy()
    assert out.shape == (x.n_w, x.n_chol + 3) and (fl.cpu().numpy() == 0).all()
    fb, E = out[:, :x.n_chol], out[:, x.n_chol:]
    ws = list(range(min(x.n_w, 6)))
    ref = o2.run(x, walkers=ws, return_G=False)
    assert_parity(dict(fb=fb, E=E), ref, walkers=ws, what=("fb", "E"))
    fb2 = trial.force_bias(pa, pb).cpu().numpy()
    E2 = trial.local_energy(pa, pb).cpu().numpy()
    assert (np.abs(fb - fb2).max(axis=1) / np.abs(fb2).max(axis=1)).max() <= TOL_REL
    assert np.abs(E - E2).max() <= TOL_E
    outh = trial.force_bias_energy_host(np.ascontiguousarray(x.phi_a), np.ascontiguousarray(x.phi_b))
    assert (np.abs(outh[:, :x.n_chol] - fb).max(axis=1) / np.abs(fb).max(axis=1)).max() <= TOL_REL
    assert np.abs(outh[:, x.n_chol:] - E).max() <= TOL_E
    trial.close()


@pytest.mark.parametrize("level", [1, 2])
def test_paths_for_windows_too_wide_for_shared_memory_tiles(torch_cuda, level):
    """The force-bias RED scatter, the energy path with Hrot / F read through L1 (level 1) and the forms that read the g
    slices through L1 as well (level 2) are what runs when a walker tile's C / Hrot / F / g do not fit in shared memory;
    no BASELINE config is that wide, so the context option MSD_OPT_NO_SMEM_TILES forces them (no environment variable)."""
    msd = _msd()
    for x, ws in ((mi.generate("small"), None), (mi.generate("sweep", n_det=3000, max_level=6, n_w=16), [0, 9, 15])):
        trial = msd.setup_from_inputs(x)
        trial.set_option(msd.MSD_OPT_NO_SMEM_TILES, level)
        got = gpu_all(torch_cuda, x, trial=trial, want_G=ws is None)
        pa = torch_cuda.tensor(x.phi_a, device="cuda")
        pb = torch_cuda.tensor(x.phi_b, device="cuda")
        fused = trial.force_bias_energy(pa, pb).cpu().numpy()
        with pytest.raises(msd.MSDError):
            trial.set_option(99, 1)
        trial.close()
        ref = o2.run(x, walkers=ws, return_G=ws is None)
        assert_parity(got, ref, walkers=ws)
        sel = np.arange(x.n_w) if ws is None else np.asarray(ws)
        assert_parity(dict(fb=fused[:, :x.n_chol], E=fused[:, x.n_chol:]), ref, walkers=sel, what=("fb", "E"))


@pytest.mark.parametrize("name,kw", [("small", {}), ("open-shell", {}), ("sweep", dict(n_det=3000, max_level=7, n_w=21))])
def test_force_bias_with_overlap_from_one_pass(torch_cuda, name, kw):
    """msd_force_bias_overlap: force bias and overlap of the same walkers from one determinant pass against the oracle and
    against the two separate calls; ragged batch, a chunked workspace (small), flags."""
    torch = torch_cuda
    msd = _msd()
    x = mi.generate(name, **kw)
    trial = msd.setup_from_inputs(x)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    fl = torch.full((x.n_w,), -1, dtype=torch.int32, device="cuda")
    fb, ov = trial.force_bias_overlap(pa, pb, flags=fl)
    fb, ov = fb.cpu().numpy(), ov.cpu().numpy()
    assert (fl.cpu().numpy() == 0).all()
    ws = list(range(min(x.n_w, 6)))
    ref = o2.run(x, walkers=ws, want=("ovlp", "greens"), return_G=False)
    assert_parity(dict(ovlp=ov, fb=fb), ref, walkers=ws, what=("ovlp", "fb"))
    ov2 = trial.overlap(pa, pb).cpu().numpy()
    fb2 = trial.force_bias(pa, pb).cpu().numpy()
    assert (np.abs(ov - ov2) / np.abs(ov2)).max() <= TOL_REL
    assert (np.abs(fb - fb2).max(axis=1) / np.abs(fb2).max(axis=1)).max() <= TOL_REL
    if name == "small":
        trial.set_workspace_limit(600 * 1024)       # one walker tile needs 0.41 MB: several chunks, the overlaps land at their offsets
        fb3, ov3 = trial.force_bias_overlap(pa, pb)
        assert (np.abs(ov3.cpu().numpy() - ov2) / np.abs(ov2)).max() <= TOL_REL
        assert (np.abs(fb3.cpu().numpy() - fb2).max(axis=1) / np.abs(fb2).max(axis=1)).max() <= TOL_REL
    with pytest.raises(ValueError):
        trial.force_bias_overlap(pa, pb, out_ovlp=torch.empty(x.n_w + 1, dtype=torch.complex128, device="cuda"))
    trial.close()


@pytest.mark.parametrize("name,kw,ws", [("small", {}, None), ("cu2o2", dict(n_w=24), [0, 7, 8, 23]),
                                        ("sweep", dict(n_det=2000, max_level=5, n_w=16), [0, 15])])
def test_alternative_dense_paths(torch_cuda, name, kw, ws):
    """The energy through the non-default dense kernels -- Lambda GEMM + dense kernel pair instead of the fused S7 kernel
    (MSD_OPT_NO_FUSED_S7), four-multiplication V GEMM instead of the three-multiplication one (MSD_OPT_NO_3M) -- against
    the oracle, and against the default path."""
    msd = _msd()
    torch = torch_cuda
    x = mi.generate(name, **kw)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    ref = o2.run(x, walkers=ws, return_G=False)
    sel = np.arange(x.n_w) if ws is None else np.asarray(ws)
    res = {}
    pure3m = ((msd.MSD_OPT_3M_MAX_COND, 10 ** 9),)      # the 3-multiplication kernel for every walker, whatever its conditioning
    for opts in ((), (msd.MSD_OPT_NO_FUSED_S7,), (msd.MSD_OPT_NO_3M,), (msd.MSD_OPT_NO_FUSED_S7, msd.MSD_OPT_NO_3M), pure3m,
                 ((msd.MSD_OPT_3M_MAX_COND, 0),)):
        trial = msd.setup_from_inputs(x)
        for o in opts:
            trial.set_option(*(o if isinstance(o, tuple) else (o, 1)))
        E = trial.local_energy(pa, pb).cpu().numpy()
        fused = trial.force_bias_energy(pa, pb).cpu().numpy()
        trial.close()
        assert np.abs(E[sel] - ref["E"]).max() <= TOL_E, opts
        assert np.abs(fused[sel, x.n_chol:] - ref["E"]).max() <= TOL_E, opts
        res[opts] = E
    for opts, E in res.items():
        # every walker of the batch, oracle-checked or not.  The pure 3-multiplication path is left out: on walkers with an
        # ill-conditioned reference block it is 4-15 x less accurate than the others, which is why
        # the default routes those walkers to the 4-multiplication kernel.
        if opts != pure3m:
            assert np.abs(E - res[()]).max() <= TOL_E, opts


@pytest.mark.parametrize("kw,ws", [(dict(n_det=3000, max_level=7, n_w=21), [0, 8, 20]),
                                   (dict(n_det=1500, max_level=10, n_w=9), [8])])
def test_high_level_kernels_both_ways(torch_cuda, kw, ws):
    """MSD_OPT_COOP_MIN_ELEMS: every bucket with a level >= 5 through the warp-cooperative kernel (threshold 0: also the
    buckets whose other spin is at level 0..4, i.e. its closed-form branch) and through the one-determinant-per-thread
    kernel (threshold 200: also levels 9-10, its runtime-k branch and CTAs below 128 threads) -- overlap, force bias
    and energy against the oracle O2, fused call included; ragged last walker tile."""
    msd = _msd()
    torch = torch_cuda
    x = mi.generate("sweep", **kw)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    ref = o2.run(x, walkers=ws, return_G=False)
    for th in (0, 200):
        trial = msd.setup_from_inputs(x)
        with pytest.raises(msd.MSDError):
            trial.set_option(msd.MSD_OPT_COOP_MIN_ELEMS, 201)
        trial.set_option(msd.MSD_OPT_COOP_MIN_ELEMS, th)
        got = dict(ovlp=trial.overlap(pa, pb).cpu().numpy(), fb=trial.force_bias(pa, pb).cpu().numpy(),
                   E=trial.local_energy(pa, pb).cpu().numpy())
        fused = trial.force_bias_energy(pa, pb).cpu().numpy()
        trial.close()
        assert_parity(got, ref, walkers=ws, what=("ovlp", "fb", "E"))
        assert_parity(dict(fb=fused[:, :x.n_chol], E=fused[:, x.n_chol:]), ref, walkers=ws, what=("fb", "E"))


def test_window_wider_than_shared_memory(torch_cuda):
    """An active window of 10 occupied x 100 virtual orbitals per spin (the paper's [Cu2O2]2+ has 16 x 92,
    PAPER.md:L303): 2000 pair indices, so neither the g slices (256 KB per walker tile) nor C / Hrot / F fit in shared
    memory, and n_v > 16 takes the scalar S7 kernel.  Every call against O2 on every walker."""
    msd = _msd()
    x = mi.wide_window()
    trial = msd.setup_from_inputs(x)
    info = trial.info()
    assert info["n_o_alpha"] * info["n_v_alpha"] + info["n_o_beta"] * info["n_v_beta"] > 1816 and info["energy_supported"]
    got = gpu_all(torch_cuda, x, trial=trial)
    pa = torch_cuda.tensor(x.phi_a, device="cuda")
    pb = torch_cuda.tensor(x.phi_b, device="cuda")
    fused = trial.force_bias_energy(pa, pb).cpu().numpy()
    trial.close()
    ref = o2.run(x)
    assert (got["flags"] == 0).all()
    assert_parity(got, ref)
    assert_parity(dict(fb=fused[:, :x.n_chol], E=fused[:, x.n_chol:]), ref, what=("fb", "E"))


def test_duplicate_determinants_are_rejected(torch_cuda):
    """Eq. 15 is an orthogonal expansion: the same determinant twice is an invalid table (MSD_EINVAL at setup), also when
    the two copies list their holes / particles in a different order or sit far apart in the list."""
    msd = _msd()
    x = mi.generate("small")
    idx = np.arange(x.n_det)
    for dup_of, at in ((5, 6), (17, x.n_det - 1), (0, 400)):
        y = x.subset_dets(np.concatenate([idx[:at], [dup_of], idx[at:]]))
        with pytest.raises(msd.MSDError) as e:
            msd.setup_from_inputs(y)
        assert e.value.code == -1 and "twice" in str(e.value)
    occa, occb = x.occa.copy(), x.occb.copy()
    occa[9], occb[9] = x.occa[3][::-1], x.occb[3]                      # same determinant, permuted occupation list
    with pytest.raises(msd.MSDError):
        msd.msd_setup_from_occ(x.N, x.n_alpha, x.n_beta, x.n_chol, x.n_det, x.h1, x.L, x.e0, occa, occb, x.ci)
    msd.setup_from_inputs(x).close()


def test_binding_validates_outputs_and_limits(torch_cuda):
    torch = torch_cuda
    msd = _msd()
    x = mi.generate("tiny")
    trial = msd.setup_from_inputs(x)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    with pytest.raises(ValueError):
        trial.force_bias(pa, pb, out=torch.empty((x.n_w, x.n_chol - 1), dtype=torch.complex128, device="cuda"))
    with pytest.raises(ValueError):
        trial.local_energy(pa, pb, out=torch.empty((x.n_w, 3), dtype=torch.complex64, device="cuda"))
    with pytest.raises(ValueError):
        trial.overlap(pa, pb, out=torch.empty(2 * x.n_w, dtype=torch.complex128, device="cuda")[::2])
    with pytest.raises(ValueError):
        trial.overlap(pa, pb, flags=torch.zeros(x.n_w - 1, dtype=torch.int32, device="cuda"))
    with pytest.raises(ValueError):
        trial.overlap_host(x.phi_a, x.phi_b, out=np.empty(x.n_w + 1, dtype=np.complex128))
    with pytest.raises(ValueError):
        trial.local_energy_host(torch.from_numpy(x.phi_a), torch.from_numpy(x.phi_b),
                                out=torch.empty((x.n_w, 3), dtype=torch.complex64))
    # two streams on one context: the second call waits for the first (one workspace per context, include/msd.h)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    fb = trial.force_bias(pa, pb, stream=s1)
    en = trial.local_energy(pa, pb, stream=s2)
    torch.cuda.synchronize()
    ref = o2.run(x, return_G=False)
    assert_parity(dict(fb=fb.cpu().numpy(), E=en.cpu().numpy()), ref, what=("fb", "E"))
    trial.close()


# ----------------------------------------------------------------------------------------------
# one phaseless-AFQMC propagation step (Eq. 5, 7-12) against oracle/propagate.py
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,kw,ws,n_taylor", [("tiny", {}, None, 6), ("open-shell", {}, None, 4), ("small", {}, None, 6),
                                                 ("cu2o2", {}, [0, 7, 8, 100, 199], 6),
                                                 # 34 + 33 electrons: more than 32 columns per walker, the orbital update's
                                                 # scalar products instead of its tensor-core form (propagate.cu prop_product)
                                                 ("small", dict(N=72, n_alpha=34, n_beta=33, A=12, n_chol=30, n_det=40, n_w=5,
                                                                max_level=3), None, 6)])
def test_propagation_step_against_oracle(torch_cuda, name, kw, ws, n_taylor):
    """msd_propagate: walkers after B(x - xbar), overlap ratio S (rel 1e-10), phase theta (abs 1e-10), importance function,
    phaseless weight update -- element by element against the numpy oracle on the same seeded fields; full batch on the
    GPU, sampled walkers in the oracle at the Cu2O2 size."""
    from oracle import propagate as op
    torch = torch_cuda
    msd = _msd()
    x = mi.generate(name, **kw)
    dt = 0.005
    rng = np.random.default_rng(11)
    fields = rng.standard_normal((x.n_w, x.n_chol))
    w0 = rng.uniform(0.5, 1.5, x.n_w)
    trial = msd.setup_from_inputs(x)
    with pytest.raises(msd.MSDError):          # no time step yet
        trial.propagate(torch.tensor(x.phi_a, device="cuda"), torch.tensor(x.phi_b, device="cuda"),
                        torch.tensor(fields, device="cuda"))
    trial.propagator_setup(dt, n_taylor, x.h1, x.L)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    wt = torch.tensor(w0, device="cuda")
    fl = torch.full((x.n_w,), -1, dtype=torch.int32, device="cuda")
    out = trial.propagate(pa, pb, torch.tensor(fields, device="cuda"), weights=wt, flags=fl).cpu().numpy()
    assert (fl.cpu().numpy() == 0).all()
    # the propagated walkers are ordinary walkers: the hot calls accept them
    ov_again = trial.overlap(pa, pb).cpu().numpy()
    trial.close()
    ref = op.step(x, fields, dt, weights=w0, n_taylor=n_taylor, walkers=ws)
    sel = np.arange(x.n_w) if ws is None else np.asarray(ws)
    pa, pb, wt = pa.cpu().numpy()[sel], pb.cpu().numpy()[sel], wt.cpu().numpy()[sel]
    out = out[sel]
    assert np.abs(pa - ref["phi_a"]).max() <= 1e-12 * np.abs(ref["phi_a"]).max()
    assert np.abs(pb - ref["phi_b"]).max() <= 1e-12 * np.abs(ref["phi_b"]).max()
    S = out[:, 0] + 1j * out[:, 1]
    assert (np.abs(S - ref["S"]) / np.abs(ref["S"])).max() <= TOL_REL
    dth = np.angle(np.exp(1j * (out[:, 2] - ref["theta"])))
    assert np.abs(dth).max() <= TOL_REL
    ovn = out[:, 4] + 1j * out[:, 5]
    assert (np.abs(ovn - ref["ovlp_new"]) / np.abs(ref["ovlp_new"])).max() <= TOL_REL
    assert (np.abs(ov_again[sel] - ref["ovlp_new"]) / np.abs(ref["ovlp_new"])).max() <= TOL_REL
    I = out[:, 6] + 1j * out[:, 7]
    assert (np.abs(I - ref["I"]) / np.abs(ref["I"])).max() <= TOL_REL
    assert np.abs(out[:, 3] - ref["I_ph"]).max() <= TOL_REL * max(1.0, np.abs(ref["I_ph"]).max())
    assert np.abs(wt - ref["w"]).max() <= TOL_REL * max(1.0, np.abs(ref["w"]).max())


def test_propagation_step_chunked_and_repeated(torch_cuda):
    """Two steps in a row under a workspace limit that forces walker chunks equal two oracle steps; dt can be changed."""
    from oracle import propagate as op
    torch = torch_cuda
    msd = _msd()
    x = mi.generate("small", n_w=21, n_det=300)
    rng = np.random.default_rng(3)
    f1, f2 = rng.standard_normal((2, x.n_w, x.n_chol))
    trial = msd.setup_from_inputs(x)
    trial.set_workspace_limit(600 * 1024)          # one walker tile needs 0.41 MB, two 0.83 MB: three chunks
    trial.propagator_setup(0.01, 6, x.h1, x.L)
    trial.propagator_setup(0.004, 6, x.h1, x.L)
    pa = torch.tensor(x.phi_a, device="cuda")
    pb = torch.tensor(x.phi_b, device="cuda")
    wt = torch.ones(x.n_w, dtype=torch.float64, device="cuda")
    trial.propagate(pa, pb, torch.tensor(f1, device="cuda"), weights=wt)
    out = trial.propagate(pa, pb, torch.tensor(f2, device="cuda"), weights=wt).cpu().numpy()
    trial.close()
    r1 = op.step(x, f1, 0.004)
    r2 = op.step(x.with_walkers(r1["phi_a"], r1["phi_b"]), f2, 0.004, weights=r1["w"])
    assert np.abs(pa.cpu().numpy() - r2["phi_a"]).max() <= 1e-11 * np.abs(r2["phi_a"]).max()
    S = out[:, 0] + 1j * out[:, 1]
    assert (np.abs(S - r2["S"]) / np.abs(r2["S"])).max() <= TOL_REL
    assert np.abs(wt.cpu().numpy() - r2["w"]).max() <= TOL_REL * np.abs(r2["w"]).max()


# ----------------------------------------------------------------------------------------------
# determinant-sharded contexts; the ranks are emulated ONE AFTER THE OTHER on this GPU
# ----------------------------------------------------------------------------------------------
class _EmulatedAllReduce:
    """Stands in for the all-reduce of `world` ranks that run in turn on one GPU.  Pass p replays the sums of the reductions
    0..p-1 (captured in earlier passes) and captures the partial buffers of reduction p; after (number of reductions + 1)
    passes every rank has seen every reduction with the full sum, which is what concurrent ranks see."""

    def __init__(self, world):
        self.world = world
        self.partial = {}                         # (reduction index, rank) -> tensor
        self.rank = 0
        self.idx = 0

    def begin(self, rank):
        self.rank, self.idx = rank, 0

    def __call__(self, t):
        k = self.idx
        self.idx += 1
        if all((k, r) in self.partial and self.partial[(k, r)] is not None for r in range(self.world)) and self.sealed > k:
            t.copy_(sum(self.partial[(k, r)] for r in range(self.world)))
        else:
            self.partial[(k, self.rank)] = t.clone()


@pytest.mark.parametrize("name,kw,world", [("small", dict(n_w=13), 2), ("sweep", dict(n_det=1500, max_level=6, n_w=9), 3)])
def test_determinant_sharded_contexts_emulated_ranks(torch_cuda, name, kw, world):
    """Every rank holds the whole trial but evaluates 1/world of every level bucket; the hook sums the partial W, C, E1nd,
    E2nd.  Overlap, force bias, energy, the fused call and a propagation step must equal the oracle (and the unsharded
    library) for every rank."""
    from oracle import propagate as op
    torch = torch_cuda
    msd = _msd()
    x = mi.generate(name, **kw)
    ref = o2.run(x, return_G=False)
    fields = np.random.default_rng(1).standard_normal((x.n_w, x.n_chol))
    pref = op.step(x, fields, 0.005)
    trials = [msd.setup_from_inputs(x, shard=(r, world)) for r in range(world)]
    for r, t in enumerate(trials):
        info = t.info()
        assert (info["shard_rank"], info["shard_world"]) == (r, world)
        t.propagator_setup(0.005, 6, x.h1, x.L)
    pa0 = torch.tensor(x.phi_a, device="cuda")
    pb0 = torch.tensor(x.phi_b, device="cuda")
    xf = torch.tensor(fields, device="cuda")

    def run_all(fn, n_reductions):
        red = _EmulatedAllReduce(world)
        outs = None
        for p in range(n_reductions + 1):
            red.sealed = p                        # reductions < p are complete and replayed
            outs = []
            for r, t in enumerate(trials):
                t.set_allreduce(red)
                red.begin(r)
                outs.append(fn(t))
            torch.cuda.synchronize()
        return outs

    for got in run_all(lambda t: t.overlap(pa0, pb0).cpu().numpy(), 1):
        assert (np.abs(got - ref["ovlp"]) / np.abs(ref["ovlp"])).max() <= TOL_REL
    for got in run_all(lambda t: t.force_bias(pa0, pb0).cpu().numpy(), 1):
        assert (np.abs(got - ref["fb"]).max(axis=1) / np.abs(ref["fb"]).max(axis=1)).max() <= TOL_REL
    for got in run_all(lambda t: t.local_energy(pa0, pb0).cpu().numpy(), 1):
        assert np.abs(got - ref["E"]).max() <= TOL_E
    for got in run_all(lambda t: t.force_bias_energy(pa0, pb0).cpu().numpy(), 1):
        assert np.abs(got[:, x.n_chol:] - ref["E"]).max() <= TOL_E
        assert (np.abs(got[:, :x.n_chol] - ref["fb"]).max(axis=1) / np.abs(ref["fb"]).max(axis=1)).max() <= TOL_REL

    def prop(t):
        pa, pb = pa0.clone(), pb0.clone()
        out = t.propagate(pa, pb, xf).cpu().numpy()
        return out, pa.cpu().numpy()
    for out, pa in run_all(prop, 2):
        S = out[:, 0] + 1j * out[:, 1]
        assert (np.abs(S - pref["S"]) / np.abs(pref["S"])).max() <= TOL_REL
        assert np.abs(pa - pref["phi_a"]).max() <= 1e-11 * np.abs(pref["phi_a"]).max()
    for t in trials:
        t.set_allreduce(None)
        t.close()
