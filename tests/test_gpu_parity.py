"""GPU parity: the CUDA path (through the C-ABI binding) against the fp64 oracle, element by
element, same seeded inputs.  Tolerances: tests/gpu_util.py (north star)."""
import numpy as np
import pytest

import oracle
from paper_1710_10789_b200 import binding, workloads as wl
from gpu_util import run_gpu, assert_parity, errors

pytestmark = pytest.mark.gpu

NT = None


def _threads():
    return oracle.max_threads()


def test_cfg1_cosine_band():
    """BASELINE config 1: closed-form band, Nk=16, W == 1 (W=NULL), 201 energies."""
    E, W, om = wl.make_inputs("cfg1")
    ref = oracle.tetra_dos(E, None, (16, 16, 16), om)
    dos, nos = run_gpu(E, None, (16, 16, 16), om)
    d, en = assert_parity(ref, dos, nos, "cfg1")
    print("cfg1 dDOS %.2e dN %.2e" % (d, en))
    # W given explicitly as ones: same result up to the order of the fp32 reductions
    dos2, nos2 = run_gpu(E, W, (16, 16, 16), om)
    assert np.allclose(dos, dos2, rtol=2e-6, atol=1e-9) and np.allclose(nos, nos2, rtol=2e-6, atol=1e-9)


def test_cfg2_tb8_nk32(cache_dir):
    """BASELINE config 2: 8-orbital model, Nk=32, 1000 energies; full element-wise comparison."""
    E, W, om = wl.make_inputs("cfg2", cache_dir)
    ref = oracle.tetra_dos(E, W, (32, 32, 32), om, windowed=True, nthreads=_threads())
    dos, nos = run_gpu(E, W, (32, 32, 32), om)
    d, en = assert_parity(ref, dos, nos, "cfg2")
    print("cfg2 dDOS %.2e dN %.2e" % (d, en))


@pytest.mark.parametrize("nk,nb,norb,nE", [
    ((2, 2, 2), 1, 1, 17),        # minimal periodic grid: every neighbour is a wrap
    ((1, 1, 1), 2, 3, 9),         # a single k-point: all four corners degenerate
    ((5, 3, 7), 3, 5, 333),       # anisotropic, ragged against every tile shape, norb not a power of 2
    ((9, 10, 11), 2, 8, 1000),
    ((17, 8, 5), 1, 2, 64),
    ((6, 6, 6), 4, 12, 257),      # norb > 8: two orbital blocks
    ((4, 4, 4), 2, 4, 1),         # a single energy
])
def test_random_small_grids(nk, nb, norb, nE):
    E, W = wl.random_bands(nk, nb, norb, seed=100 + nk[0] + nE)
    om = wl.omega_grid(-1.2, 1.3, nE)
    ref = oracle.tetra_dos(E, W, nk, om)
    for layout in (binding.TDOS_AOS, binding.TDOS_SOA):
        Ex, Wx = (E, W) if layout == binding.TDOS_AOS else wl.to_soa(E, W)
        dos, nos = run_gpu(Ex, Wx, nk, om, layout=layout)
        assert_parity(ref, dos, nos, "random %s layout %d" % (nk, layout))
    dos, nos = run_gpu(E, W, nk, om, memspace=binding.TDOS_HOST)
    assert_parity(ref, dos, nos, "random %s host" % (nk,))
    dos, nos = run_gpu(E, W, nk, om, want_nos=False)
    assert nos is None
    assert_parity(ref, dos, None, "random %s nos=NULL" % (nk,))


@pytest.mark.parametrize("kernel,variant", [("5", v) for v in range(2)] + [("3", v) for v in range(3)])
def test_every_compiled_kernel_configuration(kernel, variant, monkeypatch):
    """TDOS_KERNEL / TDOS_TILE select the kernel and the tile shape / group width / warps per block compiled into the
    library; every one of them must reproduce the oracle (tb8 model: several tiles + ragged tails; random energies,
    3 orbitals -- always tdos_main: windows spanning many passes)."""
    monkeypatch.setenv("TDOS_KERNEL", kernel)
    monkeypatch.setenv("TDOS_TILE", str(variant))
    nk = (10, 9, 7)
    E, W = wl.tb8_bands(nk, threads=1)
    om = wl.omega_grid(-6.0, 4.0, 777)
    ref = oracle.tetra_dos(E, W, nk, om, nthreads=_threads())
    with binding.Plan(nk, 8, 8, 777) as plan:
        dos, nos = run_gpu(E, W, nk, om, plan=plan)
        assert plan.last_counters()["kernel"] == int(kernel)
    assert_parity(ref, dos, nos, "tb8 kernel %s variant %d" % (kernel, variant))
    nk = (5, 6, 4)
    E, W = wl.random_bands(nk, 2, 3, seed=9)
    om = wl.omega_grid(-1.1, 1.1, 1500)
    ref = oracle.tetra_dos(E, W, nk, om)
    dos, nos = run_gpu(E, W, nk, om)
    assert_parity(ref, dos, nos, "random variant %d" % variant)


def test_ties_and_energies_on_corner_values():
    """Energies on a coarse lattice (many exact ties, flat tetrahedra) and omega exactly ON corner
    energies: the half-open interval rules (G10) decide; results must match the oracle."""
    nk, nb, norb = (6, 5, 4), 3, 3
    rng = np.random.default_rng(7)
    n = int(np.prod(nk))
    E = np.sort(rng.integers(-8, 9, (n, nb)) / 8.0, axis=1).astype(np.float32)
    W = rng.uniform(0, 1, (n, nb, norb)).astype(np.float32)
    om = (np.arange(-20, 21) / 16.0).astype(np.float32)       # every second point hits lattice values
    ref = oracle.tetra_dos(E, W, nk, om)
    dos, nos = run_gpu(E, W, nk, om)
    assert_parity(ref, dos, nos, "ties")


def test_flat_band_and_grid_outside_bands():
    nk = (4, 4, 4)
    E = np.full((64, 1), 0.25, dtype=np.float32)
    W = np.full((64, 1, 2), 0.5, dtype=np.float32)
    om = np.array([0.0, 0.25, 0.5, 0.75], dtype=np.float32)
    dos, nos = run_gpu(E, W, nk, om)
    assert not dos.any()
    assert np.allclose(nos, [[0, 0, 0.5, 0.5]] * 2, atol=1e-7)
    E, W = wl.random_bands(nk, 2, 2, seed=3)
    lo = np.array([-5.0, -4.0], dtype=np.float32)
    hi = np.array([4.0, 5.0], dtype=np.float32)
    d, n = run_gpu(E, W, nk, lo)
    assert not d.any() and not n.any()
    d, n = run_gpu(E, W, nk, hi)
    assert not d.any()
    assert np.allclose(n, W.astype(np.float64).sum(axis=(0, 1))[:, None] / 64, rtol=1e-6)


def test_nonuniform_omega_grid():
    """Any strictly increasing grid is handled exactly (index guess + exact fix-up)."""
    nk, nb, norb = (7, 7, 7), 2, 2
    E, W = wl.random_bands(nk, nb, norb, seed=21)
    rng = np.random.default_rng(1)
    om = np.unique(np.concatenate([np.linspace(-1.5, -0.5, 10), np.sort(rng.uniform(-0.5, 0.6, 150)),
                                   np.linspace(0.6, 1.5, 7)]).astype(np.float32))
    ref = oracle.tetra_dos(E, W, nk, om)
    dos, nos = run_gpu(E, W, nk, om)
    assert_parity(ref, dos, nos, "nonuniform")


def test_partial_slabs_and_finalize():
    """tetra_dos_partial over disjoint z-slabs, summed, then tetra_dos_finalize == tetra_dos
    (the multi-GPU building blocks), and each slab's share matches the oracle's cube range."""
    import torch
    nk, nb, norb, nE = (6, 5, 9), 2, 3, 200
    E, W = wl.random_bands(nk, nb, norb, seed=5)
    om = wl.omega_grid(-1.2, 1.3, nE)
    ref = oracle.tetra_dos(E, W, nk, om)
    dev = torch.device("cuda:0")
    dE, dW, dOm = (torch.from_numpy(x).to(dev) for x in (E, W, om))
    with binding.Plan(nk, nb, norb, nE) as plan:
        total = torch.zeros((3, norb, nE), dtype=torch.float64, device=dev)
        for z_lo, z_hi in ((0, 4), (4, 5), (5, 9)):
            part = torch.empty((3, norb, nE), dtype=torch.float64, device=dev)
            plan.tetra_dos_partial(dE, dW, dOm, z_lo, z_hi, part)
            total += part
        dos = torch.empty((norb, nE), device=dev)
        nos = torch.empty((norb, nE), device=dev)
        plan.tetra_dos_finalize(total, nE, dos, nos)
        torch.cuda.synchronize()
        assert_parity(ref, dos.cpu().numpy(), nos.cpu().numpy(), "slabs")
        # the same with arrays that hold only a slab's planes plus its halo plane (tetra_dos_partial_slab): equal
        # shares, AoS and SoA; the last slab's halo is plane 0
        plane = nk[0] * nk[1]
        for z_lo, z_hi in ((0, 4), (4, 5), (5, 9)):
            zs = [z % nk[2] for z in range(z_lo, z_hi + 1)]
            idx = np.concatenate([np.arange(z * plane, (z + 1) * plane) for z in zs])
            El, Wl = np.ascontiguousarray(E[idx]), np.ascontiguousarray(W[idx])
            want = torch.empty((3, norb, nE), dtype=torch.float64, device=dev)
            plan.tetra_dos_partial(dE, dW, dOm, z_lo, z_hi, want)
            for layout in (binding.TDOS_AOS, binding.TDOS_SOA):
                Ex, Wx = (El, Wl) if layout == binding.TDOS_AOS else wl.to_soa(El, Wl)
                got = torch.full((3, norb, nE), float("nan"), dtype=torch.float64, device=dev)
                plan.tetra_dos_partial_slab(torch.from_numpy(Ex).to(dev), torch.from_numpy(Wx).to(dev), dOm, z_lo, z_hi, got,
                                            layout=layout)
                torch.cuda.synchronize()
                assert torch.allclose(got, want, rtol=1e-5, atol=1e-9 * float(want.abs().max())), (z_lo, z_hi, layout)
        with pytest.raises(binding.TdosError):
            plan.tetra_dos_partial_slab(dE, dW, dOm, 4, 4, part)          # an empty slab
        # one slab against the oracle's share of the same cubes
        part = torch.empty((3, norb, nE), dtype=torch.float64, device=dev)
        plan.tetra_dos_partial(dE, dW, dOm, 4, 5, part)
        plan.tetra_dos_finalize(part, nE, dos, nos)
        torch.cuda.synchronize()
        sl = oracle.tetra_dos(E, W, nk, om, cube_range=(4 * 30, 5 * 30))
        d = np.abs(dos.cpu().numpy() - sl["dos"]).max() / ref["dos"].max()
        n = np.abs(nos.cpu().numpy() - sl["nos"]).max() / ref["nos"].max()
        assert d < 1e-5 and n < 1e-6


def test_error_codes_on_gpu():
    import torch
    nk, nb, norb, nE = (4, 4, 4), 1, 2, 16
    E, W = wl.random_bands(nk, nb, norb, seed=1)
    om = wl.omega_grid(-1, 1, nE)
    dev = torch.device("cuda:0")
    dE, dW, dOm = (torch.from_numpy(x).to(dev) for x in (E, W, om))
    dos = torch.zeros((norb, nE), device=dev)
    with binding.Plan(nk, nb, norb, nE) as plan:
        with pytest.raises(binding.TdosError) as ei:   # W == NULL needs norb == 1
            plan.tetra_dos(dE, None, dOm, dos)
        assert ei.value.code == binding.TDOS_EINVAL
        with pytest.raises(binding.TdosError):         # nE > nE_max
            plan.tetra_dos(dE, dW, torch.zeros(nE + 1, device=dev), dos)
        with pytest.raises(binding.TdosError):         # bad layout
            plan.tetra_dos(dE, dW, dOm, dos, layout=7)
        with pytest.raises(binding.TdosError):         # host mode validates omega
            bad = om.copy()
            bad[3] = bad[2]
            plan.tetra_dos(E, W, bad, np.zeros((norb, nE), dtype=np.float32), memspace=binding.TDOS_HOST)
        with pytest.raises(binding.TdosError):         # bad slab
            plan.tetra_dos_partial(dE, dW, dOm, 3, 9, torch.zeros((3, norb, nE), dtype=torch.float64, device=dev))
        assert not dos.any()                           # outputs untouched on error
        plan.tetra_dos(dE, dW, dOm, dos)               # and the plan is still usable
        torch.cuda.synchronize()
        assert dos.any()


def test_tetra_dos_simple_host_oneshot():
    E, W = wl.tb8_bands((10, 10, 10), threads=1)
    nE = 300
    om = wl.omega_grid(-6.0, 4.0, nE)
    ref = oracle.tetra_dos(E, W, (10, 10, 10), om, nthreads=_threads())
    dos = np.zeros((8, nE), dtype=np.float32)
    nos = np.zeros((8, nE), dtype=np.float32)
    binding.tetra_dos_simple(E, W, 10, 8, 8, -6.0, 4.0, nE, dos, nos)
    assert_parity(ref, dos, nos, "simple")


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times (default plan, AoS,
# device-resident; config 5 also through the HOST path it is defined on).  The windowed oracle
# (pinned against the literal one by test_P9_invariances_and_variants) computes every output here,
# so the comparison is element by element, not sampled; the kernel's exact work counters must equal
# the oracle's, and the sum rule N_m(omega_max) = (1/nk) sum_k sum_n W (P6) must hold at full size.
_REF_CACHE = {}


def _full_ref(name, cache_dir):
    """inputs and oracle result of a config, computed once per test session"""
    if name not in _REF_CACHE:
        cfg = wl.CONFIGS[name]
        E, W, om = wl.make_inputs(cfg, cache_dir)
        _REF_CACHE[name] = (E, W, om, oracle.tetra_dos(E, W, cfg.nk, om, windowed=True, nthreads=_threads()))
    return _REF_CACHE[name]


def _full_config(name, cache_dir, host=False, calls=3, expect_kernel=None):
    """`calls` calls on ONE plan, parity after each: the kernel a plan uses is picked per call on the device, so every
    call of the sequence is a result a user can get."""
    import torch
    cfg = wl.CONFIGS[name]
    E, W, om, ref = _full_ref(name, cache_dir)
    total = W.astype(np.float64).sum(axis=(0, 1)) / np.prod(cfg.nk)
    with binding.Plan(cfg.nk, cfg.nb, cfg.norb, cfg.nE) as plan:
        for call in range(calls):
            dos, nos = run_gpu(E, W, cfg.nk, om, plan=plan,
                               memspace=binding.TDOS_HOST if host else binding.TDOS_DEVICE)
            cnt = plan.last_counters()
            d, en = assert_parity(ref, dos, nos, "%s call %d" % (name, call))
            assert cnt["n_tb"] == ref["n_tb"] == 6 * int(np.prod(cfg.nk)) * cfg.nb
            assert cnt["n_eval"] == ref["n_eval"]
            if expect_kernel is not None:
                assert cnt["kernel"] == expect_kernel
            assert np.allclose(nos[:, -1], total, rtol=2e-6)
            print("%s%s call %d kernel %d dDOS %.2e dN %.2e n_eval %d" %
                  (name, " (host)" if host else "", call, cnt["kernel"], d, en, cnt["n_eval"]))
    torch.cuda.empty_cache()


def test_cfg3_full_size(cache_dir):
    _full_config("cfg3", cache_dir, expect_kernel=5)


def test_cfg4_full_size_headline(cache_dir):
    _full_config("cfg4", cache_dir, expect_kernel=5)


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_full_size_soa_layout(name, cache_dir):
    """north_star (1) names a k-major SoA layout (E[n][ik], W[n][m][ik]): the same full-size comparison with the
    inputs transposed, device mode, generation 5; work counters equal to the oracle's."""
    cfg = wl.CONFIGS[name]
    E, W, om, ref = _full_ref(name, cache_dir)
    Es, Ws = wl.to_soa(E, W)
    with binding.Plan(cfg.nk, cfg.nb, cfg.norb, cfg.nE) as plan:
        dos, nos = run_gpu(Es, Ws, cfg.nk, om, layout=binding.TDOS_SOA, plan=plan)
        cnt = plan.last_counters()
    del Es, Ws
    d, en = assert_parity(ref, dos, nos, name + " SoA")
    assert cnt["kernel"] == 5 and cnt["n_tb"] == ref["n_tb"] and cnt["n_eval"] == ref["n_eval"]
    print("%s SoA dDOS %.2e dN %.2e" % (name, d, en))


def test_cfg5_full_size_host_inputs(cache_dir):
    """windows of 3 bins: the device picks tdos_main (generation 3) on every call"""
    _full_config("cfg5", cache_dir, host=True, calls=2, expect_kernel=3)


def test_cfg5_full_size_device_resident(cache_dir):
    _full_config("cfg5", cache_dir, calls=2, expect_kernel=3)


@pytest.mark.parametrize("name,kernel", [("cfg4", 3), ("cfg5", 5)])
def test_full_size_with_the_other_kernel(name, kernel, cache_dir, monkeypatch):
    """the kernel the device would not pick for this config, forced: same tolerances at full size"""
    monkeypatch.setenv("TDOS_KERNEL", str(kernel))
    _full_config(name, cache_dir, calls=1, expect_kernel=kernel)


def test_kernel_generation_3_on_eight_orbitals(monkeypatch):
    """TDOS_KERNEL=3 forces tdos_main (the kernel used for norb < 5 or norb % 4 != 0) on 8 orbitals: same results."""
    monkeypatch.setenv("TDOS_KERNEL", "3")
    for nk, nb, norb, nE in (((9, 10, 11), 2, 8, 1000), ((6, 6, 6), 4, 12, 257)):
        E, W = wl.random_bands(nk, nb, norb, seed=100 + nk[0] + nE)
        om = wl.omega_grid(-1.2, 1.3, nE)
        ref = oracle.tetra_dos(E, W, nk, om)
        with binding.Plan(nk, nb, norb, nE) as plan:
            dos, nos = run_gpu(E, W, nk, om, plan=plan)
            assert plan.last_counters()["kernel"] == 3
        assert_parity(ref, dos, nos, "kernel 3 %s" % (nk,))
    E, W = wl.tb8_bands((12, 12, 12), threads=1)
    om = wl.omega_grid(-6.0, 4.0, 900)
    ref = oracle.tetra_dos(E, W, (12, 12, 12), om, nthreads=_threads())
    dos, nos = run_gpu(E, W, (12, 12, 12), om)
    assert_parity(ref, dos, nos, "kernel 3 tb8")


@pytest.mark.parametrize("seed", [3, 11, 29, 57])
def test_unstructured_energies_many_seeds(seed):
    """Random energies without any band continuity put tetrahedra with E1 ~ E2 ~ E3 << E4 next to the bottom of
    the spectrum, where abs(dN)/N is taken against a tiny N (G17): both kernels, several seeds."""
    for nk, nb, norb, nE in (((5, 3, 7), 3, 5, 333), ((5, 3, 7), 3, 8, 333)):
        E, W = wl.random_bands(nk, nb, norb, seed=seed)
        om = wl.omega_grid(-1.1, 1.2, nE)
        ref = oracle.tetra_dos(E, W, nk, om)
        dos, nos = run_gpu(E, W, nk, om)
        assert_parity(ref, dos, nos, "seed %d norb %d" % (seed, norb))


def test_paper_shaped_anisotropic_grid(cache_dir):
    """60 x 60 x 10 k-points, 8 bands, 1024 energies (the shapes of Table II's last row)."""
    _full_config("paper60", cache_dir)


@pytest.mark.parametrize("nk,nb,norb,nE", [
    ((4, 4, 8), 2, 8, 1),         # a single energy
    ((3, 5, 2), 1, 8, 3),         # fewer energies than a chunk of 4 bins, ragged against every tile
    ((6, 4, 16), 2, 8, 130),      # windows cross the 128-bin pass boundary
    ((2, 2, 2), 3, 16, 61),       # two orbital blocks, every neighbour is a wrap
    ((7, 6, 9), 2, 12, 515),      # second orbital block half empty (norb = 12)
])
def test_generation5_edge_cases(nk, nb, norb, nE, monkeypatch):
    """tdos_main5 (the kernel for windows of many bins when norb % 4 == 0, norb >= 5; forced here) on the degenerate
    shapes: AoS, SoA, host mode, random energies and lattice energies with omega ON the corner values (ties, G10/G11)."""
    monkeypatch.setenv("TDOS_KERNEL", "5")
    E, W = wl.random_bands(nk, nb, norb, seed=7 + nE)
    om = wl.omega_grid(-1.1, 1.2, nE)
    ref = oracle.tetra_dos(E, W, nk, om)
    with binding.Plan(nk, nb, norb, nE) as plan:
        dos, nos = run_gpu(E, W, nk, om, plan=plan)
        cnt = plan.last_counters()
    assert cnt["kernel"] == 5 and cnt["n_tb"] == ref["n_tb"] and cnt["n_eval"] == ref["n_eval"]
    assert cnt["n_eval_mid"] == ref["n_case"][1]
    assert_parity(ref, dos, nos, "gen5 %s" % (nk,))
    Es, Ws = wl.to_soa(E, W)
    dos, nos = run_gpu(Es, Ws, nk, om, layout=binding.TDOS_SOA)
    assert_parity(ref, dos, nos, "gen5 SoA %s" % (nk,))
    dos, nos = run_gpu(E, W, nk, om, memspace=binding.TDOS_HOST)
    assert_parity(ref, dos, nos, "gen5 host %s" % (nk,))
    rng = np.random.default_rng(nE)
    n = int(np.prod(nk))
    E2 = np.sort(rng.integers(-8, 9, (n, nb)) / 8.0, axis=1).astype(np.float32)
    om2 = np.unique(np.concatenate([om, (np.arange(-9, 10) / 8.0).astype(np.float32)]))[:max(nE, 1)]
    ref2 = oracle.tetra_dos(E2, W, nk, om2)
    dos, nos = run_gpu(E2, W, nk, om2)
    assert_parity(ref2, dos, nos, "gen5 ties %s" % (nk,))


@pytest.mark.parametrize("nk,nb,norb,nE", [((6, 5, 8), 2, 8, 300), ((5, 4, 3), 3, 3, 120)])
def test_complex_eigenvector_input(nk, nb, norb, nE):
    """tetra_dos_complex takes the eigenvector elements a_n^m(k) (re, im), as the paper's
    kernel does, and squares them while staging; result = tetra_dos on b = abs(a)^2."""
    import torch
    E, W = wl.random_bands(nk, nb, norb, seed=41)
    rng = np.random.default_rng(5)
    phase = rng.uniform(0, 2 * np.pi, W.shape)
    A = np.stack([np.sqrt(W) * np.cos(phase), np.sqrt(W) * np.sin(phase)], axis=-1).astype(np.float32)   # [ik][n][m][2]
    Wb = (A[..., 0].astype(np.float64) ** 2 + A[..., 1].astype(np.float64) ** 2).astype(np.float32)
    om = wl.omega_grid(-1.2, 1.3, nE)
    ref = oracle.tetra_dos(E, Wb, nk, om)
    dev = torch.device("cuda:0")
    with binding.Plan(nk, nb, norb, nE) as plan:
        for layout in (binding.TDOS_AOS, binding.TDOS_SOA):
            Ex = E if layout == binding.TDOS_AOS else np.ascontiguousarray(E.T)
            Ax = A if layout == binding.TDOS_AOS else np.ascontiguousarray(A.transpose(1, 2, 0, 3))   # [n][m][ik][2]
            dE, dA, dOm = (torch.from_numpy(np.ascontiguousarray(x)).to(dev) for x in (Ex, Ax, om))
            dos = torch.full((norb, nE), float("nan"), device=dev)
            nos = torch.full((norb, nE), float("nan"), device=dev)
            plan.tetra_dos_complex(dE, dA, dOm, dos, nos, layout=layout)
            torch.cuda.synchronize()
            assert_parity(ref, dos.cpu().numpy(), nos.cpu().numpy(), "complex layout %d" % layout)
            hdos = np.full((norb, nE), np.nan, dtype=np.float32)
            hnos = np.full((norb, nE), np.nan, dtype=np.float32)
            plan.tetra_dos_complex(Ex, Ax, om, hdos, hnos, layout=layout, memspace=binding.TDOS_HOST)
            assert_parity(ref, hdos, hnos, "complex host layout %d" % layout)
        # a real call on the same plan afterwards still works (the staging buffer only ever grows)
        hdos = np.zeros((norb, nE), dtype=np.float32)
        plan.tetra_dos(E, Wb, om, hdos, None, memspace=binding.TDOS_HOST)
        assert_parity(ref, hdos, None, "real after complex")
        with pytest.raises(binding.TdosError):
            plan.tetra_dos_complex(E, None, om, hdos, None, memspace=binding.TDOS_HOST)


@pytest.mark.parametrize("nk,nb", [((6, 5, 4), 3), ((2, 2, 2), 1), ((9, 7, 5), 2)])
def test_per_k_integration_weights(nk, nb):
    """tetra_weights (Eq. 5-7) against oracle.tetra_weights, element by element; odd and
    even numbers of energies, an energy below and above all bands, energies ON band values (ties, G10)."""
    import torch
    E, _ = wl.random_bands(nk, nb, 1, seed=23)
    n = int(np.prod(nk))
    en = np.array([-2.0, -0.7, -0.2, float(E[0, 0]), 0.1, 0.55, 3.0], dtype=np.float32)
    dev = torch.device("cuda:0")
    with binding.Plan(nk, nb, 1, 8) as plan:
        for nW in (7, 4, 1):
            for layout in (binding.TDOS_AOS, binding.TDOS_SOA):
                Ex = E if layout == binding.TDOS_AOS else np.ascontiguousarray(E.T)
                wk_ref, dwk_ref = oracle.tetra_weights(Ex, nk, en[:nW], layout=layout)
                dE, dEn = torch.from_numpy(np.ascontiguousarray(Ex)).to(dev), torch.from_numpy(en[:nW].copy()).to(dev)
                wk = torch.full((nW, nb, n), float("nan"), device=dev)
                dwk = torch.full((nW, nb, n), float("nan"), device=dev)
                plan.tetra_weights(dE, dEn, wk, dwk, layout=layout)
                torch.cuda.synchronize()
                w, d = wk.cpu().numpy().astype(np.float64), dwk.cpu().numpy().astype(np.float64)
                assert np.abs(w - wk_ref).max() <= 5e-6 / n, np.abs(w - wk_ref).max() * n
                assert np.abs(d - dwk_ref).max() <= 1e-5 * max(np.abs(dwk_ref).max(), 1e-300)
                assert not w[wk_ref == 0].any()
                wk2 = torch.full((nW, nb, n), float("nan"), device=dev)
                plan.tetra_weights(dE, dEn, wk2, None, layout=layout)        # dwk = NULL
                torch.cuda.synchronize()
                assert torch.equal(torch.nan_to_num(wk2), torch.nan_to_num(wk)) or np.allclose(wk2.cpu().numpy(), w, atol=1e-6 / n)


def test_plan_picks_kernel_per_call_on_the_device(monkeypatch):
    """Unless TDOS_KERNEL is set, a plan on 8 orbitals enqueues both main kernels and a sample of the windows, taken on
    the device at the start of every call, decides which one runs: tdos_main (one record per tetrahedron) below 7 bins
    per window, tdos_main5 above.  The same plan serves a coarse and a fine energy grid in turn; every call is checked."""
    monkeypatch.delenv("TDOS_KERNEL", raising=False)
    nk, nb, norb = (8, 8, 8), 2, 8
    E, W = wl.tb8_bands(nk, threads=1)
    E, W = np.ascontiguousarray(E[:, :nb]), np.ascontiguousarray(W[:, :nb, :])
    grids = {24: 3, 900: 5}       # coarse grid: windows of about one bin; fine grid: tens of bins
    refs = {nE: oracle.tetra_dos(E, W, nk, wl.omega_grid(-6.0, 4.0, nE)) for nE in grids}
    with binding.Plan(nk, nb, norb, 900) as plan:
        for nE in (24, 900, 24, 24, 900):
            om = wl.omega_grid(-6.0, 4.0, nE)
            dos, nos = run_gpu(E, W, nk, om, plan=plan)
            assert_parity(refs[nE], dos, nos, "adaptive nE %d" % nE)
            cnt = plan.last_counters()
            assert cnt["kernel"] == grids[nE]
            assert cnt["n_tb"] == refs[nE]["n_tb"] and cnt["n_eval"] == refs[nE]["n_eval"]
        dos, nos = run_gpu(E, W, nk, wl.omega_grid(-6.0, 4.0, 24), plan=plan, memspace=binding.TDOS_HOST)
        assert_parity(refs[24], dos, nos, "adaptive host nE 24")
        assert plan.last_counters()["kernel"] == 3
    monkeypatch.setenv("TDOS_KERNEL", "5")
    om = wl.omega_grid(-6.0, 4.0, 24)
    with binding.Plan(nk, nb, norb, 24) as plan:
        for call in range(2):
            run_gpu(E, W, nk, om, plan=plan)
            assert plan.last_counters()["kernel"] == 5


def test_plans_do_not_lower_each_others_shared_memory_limit():
    """The dynamic shared-memory limit is an attribute of the kernel function: a second plan with a small nE_max,
    created (and destroyed) after a plan with a large one, must not break the first."""
    nk, nb, norb = (8, 8, 8), 2, 8
    E, W = wl.tb8_bands(nk, threads=1)
    E, W = np.ascontiguousarray(E[:, :nb]), np.ascontiguousarray(W[:, :nb, :])
    om = wl.omega_grid(-6.0, 4.0, 4000)
    ref = oracle.tetra_dos(E, W, nk, om)
    with binding.Plan(nk, nb, norb, 4000) as plan_a:
        with binding.Plan(nk, nb, norb, 100) as plan_b:
            run_gpu(E, W, nk, wl.omega_grid(-6.0, 4.0, 100), plan=plan_b)
        dos, nos = run_gpu(E, W, nk, om, plan=plan_a)
        assert_parity(ref, dos, nos, "plan A after plan B")


def test_back_to_back_calls_on_two_streams():
    """A plan's scratch is shared by its calls: a call on another stream waits for the previous call's end, so
    asynchronous calls issued back to back on two streams give two correct results."""
    import torch
    nk, nb, norb, nE = (10, 10, 10), 3, 8, 700
    E, W = wl.random_bands(nk, nb, norb, seed=23)
    om = wl.omega_grid(-1.2, 1.3, nE)
    ref = oracle.tetra_dos(E, W, nk, om)
    E2 = (E + np.float32(0.125)).astype(np.float32)
    ref2 = oracle.tetra_dos(E2, W, nk, om)
    dev = torch.device("cuda:0")
    dE, dE2, dW, dOm = (torch.from_numpy(a).to(dev) for a in (E, E2, W, om))
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs = [(torch.empty((norb, nE), device=dev), torch.empty((norb, nE), device=dev)) for _ in range(4)]
    torch.cuda.synchronize()
    with binding.Plan(nk, nb, norb, nE) as plan:
        for i, (st, e) in enumerate(((s1, dE), (s2, dE2), (s1, dE), (s2, dE2))):
            plan.tetra_dos(e, dW, dOm, outs[i][0], outs[i][1], stream=st.cuda_stream)
        torch.cuda.synchronize()
    for i, r in enumerate((ref, ref2, ref, ref2)):
        assert_parity(r, outs[i][0].cpu().numpy(), outs[i][1].cpu().numpy(), "two streams, call %d" % i)


def test_device_mode_call_can_be_captured_in_a_cuda_graph():
    """A TDOS_DEVICE call only enqueues work (memsets, kernels, event records) on the caller's stream, so it can be
    recorded into a CUDA graph and replayed: PAPER.md:289's best case (inputs already on the GPU) inside a host loop
    that re-launches one graph per iteration.  Captured on a side stream (a) right after a call on the same stream and
    (b) right after a call on ANOTHER stream (the plan then makes the capturing stream wait for that call's end-of-call
    event); every replay sees new band energies written in place and must match the oracle.  The timing diagnostics
    (tdos_kernel_ms) are not available for captured calls; the counters are."""
    import torch
    dev = torch.device("cuda:0")
    nk, nb, norb, nE = (12, 10, 8), 8, 8, 600
    E, W = wl.tb8_bands(nk, threads=1)
    om = wl.omega_grid(-6.0, 4.0, nE)
    shifts = (0.0, 0.11, -0.23)
    refs = [oracle.tetra_dos(E + np.float32(sh), W, nk, om, nthreads=_threads()) for sh in shifts]
    dW, dOm = torch.from_numpy(W).to(dev), torch.from_numpy(om).to(dev)
    for other_stream_first in (False, True):
        dE = torch.from_numpy(E).to(dev)
        dos = torch.zeros((norb, nE), device=dev)
        nos = torch.zeros((norb, nE), device=dev)
        side = torch.cuda.Stream()
        with binding.Plan(nk, nb, norb, nE) as plan:
            with torch.cuda.stream(side):
                plan.tetra_dos(dE, dW, dOm, dos, nos, stream=side)          # warm-up on the capture stream
            torch.cuda.synchronize()
            if other_stream_first:
                plan.tetra_dos(dE, dW, dOm, dos, nos)                        # last call before the capture: current stream
                torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                plan.tetra_dos(dE, dW, dOm, dos, nos, stream=torch.cuda.current_stream())
            for sh, ref in zip(shifts, refs):
                dE.copy_(torch.from_numpy(E + np.float32(sh)))
                dos.fill_(float("nan"))
                nos.fill_(float("nan"))
                torch.cuda.synchronize()
                g.replay()
                torch.cuda.synchronize()
                assert_parity(ref, dos.cpu().numpy(), nos.cpu().numpy(), "graph replay, shift %g" % sh)
            assert plan.last_counters()["n_eval"] == refs[-1]["n_eval"]
            # an ordinary call on the same plan afterwards still works
            dE.copy_(torch.from_numpy(E))
            plan.tetra_dos(dE, dW, dOm, dos, nos)
            torch.cuda.synchronize()
            assert_parity(refs[0], dos.cpu().numpy(), nos.cpu().numpy(), "call after the graph")
            del g


@pytest.mark.parametrize("host", [False, True])
def test_orbital_selection_plus_total_paper_shape(cache_dir, host):
    """five selected orbitals of the 8-orbital model and the total DOS on the
    paper's 60 x 60 x 10 grid with 1024 energies.  Rows 0..4 must equal the oracle's rows of those orbitals, row 5 the
    sum over all eight (reading G15; linear in W, so the oracle's rows add up to it)."""
    cfg = wl.CONFIGS["paper60"]
    E, W, om, ref = _full_ref("paper60", cache_dir)
    sel = [0, 2, 3, 5, 7]
    want = {"dos": np.concatenate([ref["dos"][sel], ref["dos"].sum(axis=0, keepdims=True)]),
            "nos": np.concatenate([ref["nos"][sel], ref["nos"].sum(axis=0, keepdims=True)])}
    import torch
    with binding.Plan(cfg.nk, cfg.nb, cfg.norb, cfg.nE) as plan:
        if host:
            dos, nos = np.full((6, cfg.nE), np.nan, np.float32), np.full((6, cfg.nE), np.nan, np.float32)
            plan.tetra_dos_select(E, W, om, sel, True, dos, nos, memspace=binding.TDOS_HOST)
        else:
            dev = torch.device("cuda:0")
            dE, dW, dOm = (torch.from_numpy(a).to(dev) for a in (E, W, om))
            ddos = torch.full((6, cfg.nE), float("nan"), device=dev)
            dnos = torch.full((6, cfg.nE), float("nan"), device=dev)
            plan.tetra_dos_select(dE, dW, dOm, sel, True, ddos, dnos)
            torch.cuda.synchronize()
            dos, nos = ddos.cpu().numpy(), dnos.cpu().numpy()
        assert plan.last_counters()["kernel"] == 5      # the selection stays on the 8-row kernel
        assert_parity(want, dos, nos, "5 orbitals + total")
        # a full call on the same plan afterwards is not affected by the selection
        dos8, nos8 = run_gpu(E, W, cfg.nk, om, plan=plan)
        assert_parity(ref, dos8, nos8, "full call after a selection")


def test_orbital_selection_small_cases():
    """total alone, repeats and order, SoA, fewer than five rows on a narrow plan (generation 3), norb = 12 with total."""
    import torch
    dev = torch.device("cuda:0")
    for nk, nb, norb, sel, total in (((7, 6, 5), 2, 8, [], True), ((7, 6, 5), 2, 8, [6, 1, 1], False),
                                     ((5, 4, 6), 3, 3, [2, 0], True), ((4, 5, 3), 2, 12, [11, 0, 4, 5, 6, 7, 8, 9, 10], True)):
        nE = 300
        E, W = wl.random_bands(nk, nb, norb, seed=5 + norb)
        om = wl.omega_grid(-1.2, 1.3, nE)
        ref = oracle.tetra_dos(E, W, nk, om)
        rows = [ref["dos"][sel]] + ([ref["dos"].sum(axis=0, keepdims=True)] if total else [])
        rown = [ref["nos"][sel]] + ([ref["nos"].sum(axis=0, keepdims=True)] if total else [])
        want = {"dos": np.concatenate(rows), "nos": np.concatenate(rown)}
        nout = len(sel) + int(total)
        for layout in (binding.TDOS_AOS, binding.TDOS_SOA):
            Ex, Wx = (E, W) if layout == binding.TDOS_AOS else wl.to_soa(E, W)
            dE, dW, dOm = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (Ex, Wx, om))
            ddos = torch.full((nout, nE), float("nan"), device=dev)
            dnos = torch.full((nout, nE), float("nan"), device=dev)
            with binding.Plan(nk, nb, norb, nE) as plan:
                plan.tetra_dos_select(dE, dW, dOm, sel, total, ddos, dnos, layout=layout)
                torch.cuda.synchronize()
            assert_parity(want, ddos.cpu().numpy(), dnos.cpu().numpy(), "select %s total %s norb %d" % (sel, total, norb))
    with binding.Plan((4, 4, 4), 2, 8, 10) as plan:
        with pytest.raises(binding.TdosError):
            plan.tetra_dos_select(dE, dW, dOm, [8], False, ddos, dnos)        # orbital out of range
        with pytest.raises(binding.TdosError):
            plan.tetra_dos_select(dE, dW, dOm, [], False, ddos, dnos)         # nothing asked for


@pytest.mark.parametrize("host", [False, True])
def test_all_eight_orbitals_plus_total_on_an_eight_orbital_plan(cache_dir, host):
    """Nine rows (every orbital of the 8-orbital model and the total) on a norb == 8 plan: one row more than the
    compile-time 8-row kernel holds, so the plan switches to the same tile with a run-time row count (12 padded rows);
    still generation 5 (round-2 advisor finding: the rows came back scrambled)."""
    import torch
    cfg = wl.CONFIGS["paper60"]
    E, W, om, ref = _full_ref("paper60", cache_dir)
    sel = [3, 0, 1, 2, 7, 6, 5, 4]
    want = {"dos": np.concatenate([ref["dos"][sel], ref["dos"].sum(axis=0, keepdims=True)]),
            "nos": np.concatenate([ref["nos"][sel], ref["nos"].sum(axis=0, keepdims=True)])}
    with binding.Plan(cfg.nk, cfg.nb, cfg.norb, cfg.nE) as plan:
        if host:
            dos, nos = np.full((9, cfg.nE), np.nan, np.float32), np.full((9, cfg.nE), np.nan, np.float32)
            plan.tetra_dos_select(E, W, om, sel, True, dos, nos, memspace=binding.TDOS_HOST)
        else:
            dev = torch.device("cuda:0")
            dE, dW, dOm = (torch.from_numpy(a).to(dev) for a in (E, W, om))
            ddos = torch.full((9, cfg.nE), float("nan"), device=dev)
            dnos = torch.full((9, cfg.nE), float("nan"), device=dev)
            plan.tetra_dos_select(dE, dW, dOm, sel, True, ddos, dnos)
            torch.cuda.synchronize()
            dos, nos = ddos.cpu().numpy(), dnos.cpu().numpy()
        assert plan.last_counters()["kernel"] == 5
        assert_parity(want, dos, nos, "8 orbitals + total")
        dos8, nos8 = run_gpu(E, W, cfg.nk, om, plan=plan)          # the 8-row kernel again
        assert_parity(ref, dos8, nos8, "full call after 9 rows")


def test_orbital_index_above_127():
    """The selection is kept in 16 bits: orbital 130 of a 132-orbital problem (round-2 advisor finding: an 8-bit
    field wrapped negative and read out of bounds)."""
    import torch
    dev = torch.device("cuda:0")
    nk, nb, norb, nE = (3, 3, 2), 1, 132, 40
    E, W = wl.random_bands(nk, nb, norb, seed=132)
    om = wl.omega_grid(-1.2, 1.3, nE)
    ref = oracle.tetra_dos(E, W, nk, om)
    sel = [130, 5, 127, 128]
    want = {"dos": np.concatenate([ref["dos"][sel], ref["dos"].sum(axis=0, keepdims=True)]),
            "nos": np.concatenate([ref["nos"][sel], ref["nos"].sum(axis=0, keepdims=True)])}
    dE, dW, dOm = (torch.from_numpy(a).to(dev) for a in (E, W, om))
    ddos = torch.full((5, nE), float("nan"), device=dev)
    dnos = torch.full((5, nE), float("nan"), device=dev)
    with binding.Plan(nk, nb, norb, nE) as plan:
        plan.tetra_dos_select(dE, dW, dOm, sel, True, ddos, dnos)
        torch.cuda.synchronize()
        assert_parity(want, ddos.cpu().numpy(), dnos.cpu().numpy(), "orbital 130")
        with pytest.raises(binding.TdosError):
            plan.tetra_dos_select(dE, dW, dOm, [132], False, ddos, dnos)


def test_fp64_accumulation_reaches_the_output_rounding_floor(cache_dir):
    """with tdos_plan_set_accumulation(TDOS_ACC_FP64) the single-precision corner
    weights are summed in fp64 everywhere.  On the band-structure configs the result then agrees with the fp64 oracle to
    the rounding of the fp32 OUTPUT arrays (6e-8): tolerance 1.5e-7 on both DOS and N, tighter than the fp32 mode reaches
    (2e-7 .. 3e-7 on N); switching back restores the default kernels."""
    for name in ("cfg2", "cfg3"):
        cfg = wl.CONFIGS[name]
        E, W, om, ref = _full_ref(name, cache_dir)
        with binding.Plan(cfg.nk, cfg.nb, cfg.norb, cfg.nE) as plan:
            plan.set_accumulation(True)
            dos, nos = run_gpu(E, W, cfg.nk, om, plan=plan)
            cnt = plan.last_counters()
            d64, n64, zero_ok = errors(ref, dos, nos)
            assert cnt["kernel"] == 3 and cnt["n_tb"] == ref["n_tb"] and cnt["n_eval"] == ref["n_eval"]
            assert zero_ok and d64 <= 1.5e-7 and n64 <= 1.5e-7, (name, d64, n64)
            dos_h, nos_h = run_gpu(E, W, cfg.nk, om, plan=plan, memspace=binding.TDOS_HOST)
            dh, nh, _ = errors(ref, dos_h, nos_h)
            assert dh <= 1.5e-7 and nh <= 1.5e-7
            plan.set_accumulation(False)
            dos, nos = run_gpu(E, W, cfg.nk, om, plan=plan)
            d32, n32 = assert_parity(ref, dos, nos, name + " fp32 again")
            assert plan.last_counters()["kernel"] == 5
            assert n64 < n32
        print("%s fp64 accumulation dDOS %.2e dN %.2e (fp32: %.2e %.2e)" % (name, d64, n64, d32, n32))


def _fp64_shares_vs_oracle(plan, E, W, nk, om, ref):
    """tetra_dos_partial over the whole grid: the raw fp64 sums, turned into DOS and N in numpy fp64 exactly as
    tetra_dos_finalize does (V * part[0]; V * (part[1] + inclusive prefix of part[2])) -- no fp32 rounding anywhere"""
    import torch
    dev = torch.device("cuda:0")
    norb = 1 if W is None else W.shape[2]
    dE, dOm = torch.from_numpy(E).to(dev), torch.from_numpy(om).to(dev)
    dW = None if W is None else torch.from_numpy(W).to(dev)
    part = torch.full((3, norb, len(om)), float("nan"), dtype=torch.float64, device=dev)
    plan.tetra_dos_partial(dE, dW, dOm, 0, nk[2], part)
    torch.cuda.synchronize()
    P = part.cpu().numpy()
    V = 1.0 / (24.0 * float(np.prod(nk)))
    dos, nos = V * P[0], V * (P[1] + np.cumsum(P[2], axis=1))
    ed = np.abs(dos - ref["dos"]).max() / ref["dos"].max()
    pos = ref["nos"] > 0
    en = (np.abs(nos - ref["nos"])[pos] / ref["nos"][pos]).max()
    assert not nos[~pos].any()
    return ed, en


def test_all_fp64_mode_agrees_with_the_oracle_to_1e_12(cache_dir):
    """PAPER.md:271 "one can in principle switch to double precision": with TDOS_ACC_FP64_ALL the corner weights are
    double precision too, so the fp64 shares of tetra_dos_partial must agree with the fp64 oracle far below single
    precision: 1e-12 on config 2 (DOS relative to its maximum, N relative wherever N > 0; measured 2e-15), against
    2e-8 .. 4e-8 with fp32 weights.  Unstructured random energies (nearly degenerate tetrahedra): 1e-11 (measured 4e-15).  The fp32 outputs of tetra_dos in this
    mode carry only their own rounding (1.5e-7)."""
    cfg = wl.CONFIGS["cfg2"]
    E, W, om, ref = _full_ref("cfg2", cache_dir)
    with binding.Plan(cfg.nk, cfg.nb, cfg.norb, cfg.nE) as plan:
        plan.set_accumulation(True)
        d1, n1 = _fp64_shares_vs_oracle(plan, E, W, cfg.nk, om, ref)          # fp32 weights, fp64 sums
        plan.set_accumulation(True, weights_fp64=True)
        d2, n2 = _fp64_shares_vs_oracle(plan, E, W, cfg.nk, om, ref)
        assert plan.last_counters()["kernel"] == 3
        dos, nos = run_gpu(E, W, cfg.nk, om, plan=plan)
        d3, n3, zero_ok = errors(ref, dos, nos)
        plan.set_accumulation(False)
        dos, nos = run_gpu(E, W, cfg.nk, om, plan=plan)
        assert_parity(ref, dos, nos, "fp32 again")
    print("cfg2 fp64 shares: fp32 weights dDOS %.2e dN %.2e; fp64 weights dDOS %.2e dN %.2e; fp32 outputs %.2e %.2e"
          % (d1, n1, d2, n2, d3, n3))
    assert d2 <= 1e-12 and n2 <= 1e-12, (d2, n2)
    assert d1 > 10 * d2 and n1 > 10 * n2            # the mode does what it says: the fp32 weights were the floor
    assert zero_ok and d3 <= 1.5e-7 and n3 <= 1.5e-7
    for nk, nb, norb, nE in (((5, 3, 7), 3, 8, 333), ((6, 5, 4), 2, 3, 200), ((3, 4, 3), 1, 1, 64)):
        E, W = wl.random_bands(nk, nb, norb, seed=41 + norb)
        if norb == 1:
            W = None
        om = wl.omega_grid(-1.1, 1.2, nE)
        ref = oracle.tetra_dos(E, W, nk, om)
        with binding.Plan(nk, nb, norb, nE) as plan:
            plan.set_accumulation(binding.TDOS_ACC_FP64_ALL)
            d, n = _fp64_shares_vs_oracle(plan, E, W, nk, om, ref)
        print("random %s fp64 weights dDOS %.2e dN %.2e" % (nk, d, n))
        assert d <= 1e-11 and n <= 1e-11, (nk, d, n)


@pytest.mark.parametrize("nk,nb,norb,nE", [((5, 3, 7), 3, 8, 333), ((6, 5, 4), 2, 3, 200), ((4, 4, 5), 2, 12, 150), ((3, 4, 3), 1, 1, 64)])
def test_fp64_accumulation_on_unstructured_energies(nk, nb, norb, nE):
    """every orbital-block width, selection + total, W = NULL: north-star tolerances (the error left is that of the
    single-precision weights at nearly degenerate tetrahedra), and never worse than 1.2 x the fp32 mode"""
    E, W = wl.random_bands(nk, nb, norb, seed=41 + norb)
    if norb == 1:
        W = None
    om = wl.omega_grid(-1.1, 1.2, nE)
    ref = oracle.tetra_dos(E, W, nk, om)
    with binding.Plan(nk, nb, norb, nE) as plan:
        dos, nos = run_gpu(E, W, nk, om, plan=plan)
        d32, n32 = assert_parity(ref, dos, nos, "fp32")
        plan.set_accumulation(True)
        dos, nos = run_gpu(E, W, nk, om, plan=plan)
        d64, n64 = assert_parity(ref, dos, nos, "fp64")
        assert n64 <= 1.2 * n32 + 1e-9 and d64 <= 1.2 * d32 + 1e-9
        if norb >= 3:
            import torch
            dev = torch.device("cuda:0")
            dE, dW, dOm = (torch.from_numpy(a).to(dev) for a in (E, W, om))
            ddos = torch.full((3, nE), float("nan"), device=dev)
            dnos = torch.full((3, nE), float("nan"), device=dev)
            plan.tetra_dos_select(dE, dW, dOm, [2, 0], True, ddos, dnos)
            torch.cuda.synchronize()
            want = {"dos": np.concatenate([ref["dos"][[2, 0]], ref["dos"].sum(axis=0, keepdims=True)]),
                    "nos": np.concatenate([ref["nos"][[2, 0]], ref["nos"].sum(axis=0, keepdims=True)])}
            assert_parity(want, ddos.cpu().numpy(), dnos.cpu().numpy(), "fp64 select")


@pytest.mark.parametrize("kernel", ["3", "5"])
def test_many_energies_no_shared_memory_copy_of_omega(kernel, monkeypatch):
    """30 000 energies: the block-wide copy of omega no longer fits beside the warps' slices (the kernels read the
    global array), windows span hundreds of bins and many 128-bin passes; norb = 16 (two orbital blocks)."""
    monkeypatch.setenv("TDOS_KERNEL", kernel)
    nk, nb, norb, nE = (6, 5, 4), 2, 16, 30000
    E, W = wl.random_bands(nk, nb, norb, seed=77)
    om = wl.omega_grid(-1.2, 1.3, nE)
    ref = oracle.tetra_dos(E, W, nk, om, windowed=True)
    with binding.Plan(nk, nb, norb, nE) as plan:
        dos, nos = run_gpu(E, W, nk, om, plan=plan)
        cnt = plan.last_counters()
    assert cnt["kernel"] == int(kernel) and cnt["n_eval"] == ref["n_eval"]
    assert_parity(ref, dos, nos, "30000 energies, kernel " + kernel)
