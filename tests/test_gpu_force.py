"""GPU parity of gint_force_stress (Eq. 4 / Eq. 5; reading R15) against the CPU oracle, through the C ABI.
Bar: max|dF| / max|F| <= 1e-10 and max|dsigma| / max|sigma| <= 1e-10 (the north_star tolerance of H and rho, carried over)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2409_09399_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-10


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _run(torch, w, V, D, flags=0, stress=True):
    from paper_2409_09399_b200.gint import Gint
    g = Gint.from_workload(w, flags=flags)
    F, sigma = g.force_stress(torch.from_numpy(V).cuda(), torch.from_numpy(D).cuda(), stress=stress)
    F2, sigma2 = g.force_stress(torch.from_numpy(V).cuda(), torch.from_numpy(D).cuda(), stress=stress)
    t = g.force_time()
    g.close()
    assert t > 0
    F, F2 = F.cpu().numpy(), F2.cpu().numpy()
    assert np.abs(F2 - F).max() <= 1e-13 * np.abs(F).max()          # repeatable to rounding (floating-point atomics)
    return F, (sigma.cpu().numpy() if stress else None)


def _rel(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


@pytest.mark.parametrize("shape", [None, (3, 3, 5), (8, 8, 8), (1, 1, 1)])
def test_cfg0_force_and_stress(torch_cuda, shape):
    """8-atom diamond: atoms sit on mesh points (the nucleus rule of the gradient), periodic images, ragged batch shapes."""
    from paper_2409_09399_b200.gint import batch_flag
    w = W.make_workload(0)
    pl = O.pairs(w)
    V = W.make_potential(w)
    D = W.make_density_blocks(w, *pl) + 0.3 * np.random.default_rng(8).standard_normal(int(pl[3][-1]))    # no symmetry of D assumed
    F, sigma = _run(torch_cuda, w, V, D, flags=batch_flag(*shape) if shape else 0)
    F_or, s_or = O.force_stress(w, V, D, pl)
    assert _rel(F, F_or) <= TOL and _rel(sigma, s_or) <= TOL


def test_cfg1_graphene_force_and_stress(torch_cuda):
    w = W.make_workload(1)
    pl = O.pairs(w)
    V = W.make_potential(w)
    D = W.make_density_blocks(w, *pl)
    F, sigma = _run(torch_cuda, w, V, D)
    F_or, s_or = O.force_stress(w, V, D, pl)
    assert _rel(F, F_or) <= TOL and _rel(sigma, s_or) <= TOL


def test_skew_two_species_force_and_stress(torch_cuda):
    b1 = W.make_basis(4.0, shells=((0, 0.7), (1, 0.5), (2, 0.45)))
    b2 = W.make_basis(3.0, shells=((0, 0.9), (0, 0.3), (1, 0.6)))
    basis = W.Basis(2, np.array([3, 3], np.int32), np.concatenate([b1.shell_l, b2.shell_l]),
                    np.array([4.0, 3.0]), W.DR, np.concatenate([b1.n_knot, b2.n_knot]),
                    np.concatenate([b1.tab_y, b2.tab_y]), np.concatenate([b1.tab_y2, b2.tab_y2]))
    cell = np.array([[5.0, 0.3, 0.0], [1.7, 4.6, 0.2], [0.4, -0.5, 5.5]])
    pos = np.array([[0.1, 0.2, 0.3], [2.5, 2.0, 1.0], [7.9, -1.0, 6.0], [3.3, 3.9, 4.4]])
    w = W.Workload("skew", 90, cell, np.array([17, 19, 23], np.int32), np.array([0, 1, 1, 0], np.int32), pos, basis)
    pl = O.pairs(w)
    rng = np.random.default_rng(12)
    V = rng.standard_normal(w.n_points); D = rng.standard_normal(int(pl[3][-1]))
    F, sigma = _run(torch_cuda, w, V, D)
    F_or, s_or = O.force_stress(w, V, D, pl)
    assert _rel(F, F_or) <= TOL and _rel(sigma, s_or) <= TOL
    # no stress wanted: same forces
    F_only, none = _run(torch_cuda, w, V, D, stress=False)
    assert none is None and np.abs(F_only - F).max() <= 1e-13 * np.abs(F).max()


def _sampled_forces(torch, cfg, n_atoms, flag_sets=(0,)):
    """Full-size workload: the forces of a stratified sample of atoms (first, last, random; the oracle computes any atom alone), from
    the library initialised with each entry of flag_sets (default batch shape, GINT_FLAG_TUNE as bench.py passes it, a forced shape)."""
    w = W.make_workload(cfg)
    pl = O.pairs(w)
    V = W.make_potential(w)
    D = W.make_density_blocks(w, *pl)
    rng = np.random.default_rng([2409, 9399, cfg, 78])
    sel = np.unique(np.concatenate([[0, w.n_atoms - 1], rng.integers(0, w.n_atoms, n_atoms)])).astype(np.int64)
    Fs = [_run(torch, w, V, D, flags=flags, stress=False)[0] for flags in flag_sets]
    F_or, _ = O.force_stress(w, V, D, pl, sel=sel)
    for flags, F in zip(flag_sets, Fs):
        err = float(np.abs(F[sel] - F_or[sel]).max() / np.abs(F).max())
        assert err <= TOL, f"cfg{cfg} flags={flags:#x} force parity on {len(sel)} atoms {err:.3e}"
    # (no net-force check: V carries seeded noise per mesh point, so E is not invariant under a rigid shift of the atoms)


def test_cfg2_bulk_sampled_forces(torch_cuda):
    _sampled_forces(torch_cuda, 2, 24)


def test_cfg3_tbg_sampled_forces(torch_cuda):
    _sampled_forces(torch_cuda, 3, 48)


def test_cfg5_mixed_species_sampled_forces(torch_cuda):
    _sampled_forces(torch_cuda, 5, 48)


def test_cfg4_tbg_headline_sampled_forces(torch_cuda):
    """As bench.py initialises the headline workload (GINT_FLAG_TUNE), and with the 4x8x16 shape forced."""
    from paper_2409_09399_b200.gint import FLAG_TUNE, batch_flag
    _sampled_forces(torch_cuda, 4, 48, flag_sets=(FLAG_TUNE, batch_flag(4, 8, 16)))


def test_dense_multi_group_cell_force_and_all_nine_stress_components(torch_cuda):
    """64-atom bulk diamond (2 x 2 x 2 cells, rc 7, mesh 67^3: ragged last batches on every axis): the largest dense cell whose full
    stress the oracle can afford.  Its batches hold several groups of atoms, so the stress (Eq. 5) crosses group
    boundaries and batch tails here, not only on the few-atom cells; D carries no mirror symmetry.  Two batch shapes."""
    from paper_2409_09399_b200.gint import Gint, batch_flag
    cell, pos = W.diamond(2)
    w = W.Workload("diamond 2x2x2 (64 atoms), rc 7", 97, np.ascontiguousarray(cell), W._mesh_for(cell), np.zeros(len(pos), np.int32),
                   np.ascontiguousarray(pos), W.make_basis(7.0))
    pl = O.pairs(w)
    V = W.make_potential(w)
    D = W.make_density_blocks(w, *pl) + 0.3 * np.random.default_rng(14).standard_normal(int(pl[3][-1]))
    g = Gint.from_workload(w)
    st = g.stats()
    g.close()
    assert st["max_nb"] > 8, "the cell is meant to need several atom groups per batch"
    F_or, s_or = O.force_stress(w, V, D, pl)
    assert np.abs(s_or).min() > 1e-4 * np.abs(s_or).max()          # all nine components carry signal
    for flags in (0, batch_flag(4, 8, 16)):
        F, sigma = _run(torch_cuda, w, V, D, flags=flags)
        assert _rel(F, F_or) <= TOL and _rel(sigma, s_or) <= TOL, f"flags={flags:#x}"


def test_force_many_orbitals_and_crowded_batches(torch_cuda):
    """A 28-orbital species beside a 4-orbital one (rows of an atom longer than a warp's share; blocks of unequal shape), and the dense
    diamond cell with rc = 8.5 whose batches hold up to 96 atom images: the force kernel's shared memory grows with the orbitals of a
    batch -- either it fits and the result is exact, or the call fails loudly with GINT_ERR_UNSUPPORTED (never a wrong result); with
    GINT_FLAG_FORCE gint_init picks a batch shape the force kernel supports, and both cells are checked against the oracle."""
    from paper_2409_09399_b200.gint import GintError
    torch = torch_cuda
    big = W.make_basis(4.5, shells=((0, 0.8), (0, 0.4), (0, 0.2), (1, 0.7), (1, 0.35), (1, 0.2), (2, 0.6), (2, 0.3), (2, 0.2), (0, 0.12)))
    small = W.make_basis(4.0, shells=((0, 0.5), (1, 0.4)))
    basis = W.concat_bases([big, small])
    rng = np.random.default_rng(31)
    cell = np.array([[6.0, 0.0, 0.0], [0.5, 5.5, 0.0], [0.0, 0.3, 6.5]])
    pos = rng.uniform(0, 1, (14, 3)) @ cell
    species = np.array([0, 0, 1, 0, 1, 0, 0, 1, 0, 0, 1, 0, 0, 1], np.int32)
    w = W.Workload("many-orbitals", 96, cell, np.array([20, 18, 22], np.int32), species, pos, basis)
    w0 = W.make_workload(0)
    wd = W.Workload("dense", 94, w0.cell, np.array([16, 16, 16], np.int32), w0.atom_species, w0.atom_pos, W.make_basis(8.5))
    from paper_2409_09399_b200.gint import FLAG_FORCE
    for wl in (w, wd):
        pl = O.pairs(wl)
        V = rng.standard_normal(wl.n_points); D = rng.standard_normal(int(pl[3][-1]))
        F_or, s_or = O.force_stress(wl, V, D, pl)
        ran = []
        for flags in (0, FLAG_FORCE):
            try:
                F, sigma = _run(torch, wl, V, D, flags=flags)
            except GintError as e:
                # only the batch shape chosen for gint_vlocal / gint_rho alone may be too big for the force kernel, and it says so
                assert flags == 0 and "shared memory" in str(e) and "GINT_FLAG_FORCE" in str(e), str(e)
                continue
            assert _rel(F, F_or) <= TOL and _rel(sigma, s_or) <= TOL
            ran.append(flags)
        print(f"gint_force_stress on {wl.name!r}: ran with flags {ran}")
        assert FLAG_FORCE in ran, f"{wl.name}: GINT_FLAG_FORCE must pick a batch shape the force kernel supports"
