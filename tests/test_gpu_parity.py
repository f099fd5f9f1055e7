"""GPU parity: libgint.so (through the C ABI, via the ctypes binding) against the CPU oracle, element by element,
on the same seeded inputs.  Bar (BASELINE.json north_star): max|dH|/max|H| <= 1e-10, max|drho|/max|rho| <= 1e-10.
The pair list is integer work: bit-exact.
"""
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


def _gint(w, flags=0):
    from paper_2409_09399_b200.gint import Gint
    return Gint.from_workload(w, flags=flags)


def _rel(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def _check_pairs(g, plist):
    A, B, R, off = g.pairs()
    oA, oB, oR, ooff = plist
    assert np.array_equal(A, oA) and np.array_equal(B, oB) and np.array_equal(R, oR) and np.array_equal(off, ooff)


def _full_parity(torch, w, flags=0, seed_extra=None):
    plist = O.pairs(w)
    g = _gint(w, flags)
    _check_pairs(g, plist)
    V = W.make_potential(w)
    D = W.make_density_blocks(w, *plist)
    if seed_extra is not None:       # break the symmetry of D: the library must honour all ordered blocks
        D = D + 0.3 * np.random.default_rng(seed_extra).standard_normal(D.size)
    H_or = O.vlocal(w, V, plist)
    rho_or = O.rho(w, D, plist)
    H = g.vlocal(torch.from_numpy(V).cuda()).cpu().numpy()
    rho = g.rho(torch.from_numpy(D).cuda()).cpu().numpy()
    eH, er = _rel(H, H_or), _rel(rho, rho_or)
    st = g.stats()
    g.close()
    assert eH <= TOL, f"H parity {eH:.3e}"
    assert er <= TOL, f"rho parity {er:.3e}"
    return st


def test_cfg0_full(torch_cuda):
    st = _full_parity(torch_cuda, W.make_workload(0))
    assert st["n_batch_empty"] == 0


def test_cfg0_nonsymmetric_D(torch_cuda):
    _full_parity(torch_cuda, W.make_workload(0), seed_extra=7)


@pytest.mark.parametrize("shape", [(2, 2, 2), (3, 3, 5), (5, 2, 3), (1, 1, 1), (4, 2, 7), (8, 8, 16), (3, 5, 13), (8, 8, 8)])
def test_cfg0_batch_shapes(torch_cuda, shape):
    """Ragged edge batches (24 is not a multiple of 5 or 7) and other batch shapes give the same result."""
    from paper_2409_09399_b200.gint import batch_flag
    st = _full_parity(torch_cuda, W.make_workload(0), flags=batch_flag(*shape))
    assert (st["batch_bx"], st["batch_by"], st["batch_bz"]) == shape


def test_cfg1_full(torch_cuda):
    st = _full_parity(torch_cuda, W.make_workload(1))
    assert st["n_batch_empty"] > 0          # vacuum


def test_skew_cell_two_species(torch_cuda):
    """Non-orthogonal cell, two species with different rc / shell sets, atoms outside the home cell, self images."""
    torch = torch_cuda
    b1 = W.make_basis(4.0, shells=((0, 0.7), (1, 0.5), (2, 0.45)))
    b2 = W.make_basis(3.0, shells=((0, 0.9), (0, 0.3), (1, 0.6)))
    basis = W.Basis(2, np.array([3, 3], np.int32), np.concatenate([b1.shell_l, b2.shell_l]),
                    np.array([4.0, 3.0]), W.DR, np.concatenate([b1.n_knot, b2.n_knot]),
                    np.concatenate([b1.tab_y, b2.tab_y]), np.concatenate([b1.tab_y2, b2.tab_y2]))
    cell = np.array([[5.0, 0.3, 0.0], [1.7, 4.6, 0.2], [0.4, -0.5, 5.5]])
    pos = np.array([[0.1, 0.2, 0.3], [2.5, 2.0, 1.0], [7.9, -1.0, 6.0], [3.3, 3.9, 4.4]])
    w = W.Workload("skew", 90, cell, np.array([17, 19, 23], np.int32), np.array([0, 1, 1, 0], np.int32), pos, basis)
    plist = O.pairs(w)
    g = _gint(w)
    _check_pairs(g, plist)
    rng = np.random.default_rng(11)
    V = rng.standard_normal(w.n_points)
    D = rng.standard_normal(int(plist[3][-1]))
    H = g.vlocal(torch.from_numpy(V).cuda()).cpu().numpy()
    rho = g.rho(torch.from_numpy(D).cuda()).cpu().numpy()
    g.close()
    assert _rel(H, O.vlocal(w, V, plist)) <= TOL
    assert _rel(rho, O.rho(w, D, plist)) <= TOL


def test_host_entry_points(torch_cuda):
    torch = torch_cuda
    w = W.make_workload(0)
    plist = O.pairs(w)
    g = _gint(w)
    V = W.make_potential(w)
    D = W.make_density_blocks(w, *plist)
    H = np.empty(g.n_values)
    rho = torch.empty(g.n_points, dtype=torch.float64).pin_memory()
    g.vlocal_host(V, H)
    g.rho_host(torch.from_numpy(D).pin_memory(), rho)
    g.close()
    assert _rel(H, O.vlocal(w, V, plist)) <= TOL
    assert _rel(rho.numpy(), O.rho(w, D, plist)) <= TOL


def test_many_waves_and_chunked_host_copies(torch_cuda):
    """A small orbital-value scratch (GINT_FLAG_PHI_CAP_MB of gint_init) cuts cfg1 into many waves, as the headline workload is cut into
    20: the device path, and the host entry points whose copies of V / rho run in per-wave chunks on a copy stream beside the kernels,
    must give the same exact results (also with a batch shape whose planes do not line up with the waves)."""
    from paper_2409_09399_b200.gint import batch_flag, phi_cap_flag
    torch = torch_cuda
    w = W.make_workload(1)
    plist = O.pairs(w)
    V = W.make_potential(w)
    D = W.make_density_blocks(w, *plist)
    H_or, rho_or = O.vlocal(w, V, plist), O.rho(w, D, plist)
    for flags in (0, batch_flag(3, 8, 16)):
        g = _gint(w, flags | phi_cap_flag(24))
        assert g.stats()["n_waves"] >= 8
        H = g.vlocal(torch.from_numpy(V).cuda()).cpu().numpy()
        rho = g.rho(torch.from_numpy(D).cuda()).cpu().numpy()
        H_h = torch.empty(g.n_values, dtype=torch.float64).pin_memory(); rho_h = torch.full((g.n_points,), np.nan, dtype=torch.float64).pin_memory()
        g.vlocal_host(torch.from_numpy(V).pin_memory(), H_h)
        g.rho_host(torch.from_numpy(D).pin_memory(), rho_h)
        g.close()
        assert _rel(H, H_or) <= TOL and _rel(rho, rho_or) <= TOL
        assert _rel(H_h.numpy(), H_or) <= TOL and _rel(rho_h.numpy(), rho_or) <= TOL


def test_empty_and_single_atom(torch_cuda):
    torch = torch_cuda
    basis = W.make_basis(5.0)
    cell = np.eye(3) * 30.0
    # no atoms at all: H is empty, rho is zero
    w0 = W.Workload("empty", 91, cell, np.array([12, 12, 12], np.int32), np.zeros(0, np.int32), np.zeros((0, 3)), basis)
    g = _gint(w0)
    assert g.n_pairs == 0 and g.n_values == 0
    rho = g.rho(torch.zeros(0, dtype=torch.float64, device="cuda")).cpu().numpy()
    assert np.all(rho == 0)
    g.close()
    # one atom in a big box: one on-site block
    w1 = W.Workload("single", 92, cell, np.array([40, 40, 40], np.int32), np.zeros(1, np.int32), np.array([[3.0, 29.0, 15.0]]), basis)
    plist = O.pairs(w1)
    g = _gint(w1)
    _check_pairs(g, plist)
    assert g.n_pairs == 1
    V = np.random.default_rng(3).standard_normal(w1.n_points)
    D = np.random.default_rng(4).standard_normal(169)
    H = g.vlocal(torch.from_numpy(V).cuda()).cpu().numpy()
    rho = g.rho(torch.from_numpy(D).cuda()).cpu().numpy()
    g.close()
    assert _rel(H, O.vlocal(w1, V, plist)) <= TOL
    assert _rel(rho, O.rho(w1, D, plist)) <= TOL


# ---------------------------------------------------------------------------------------------------------------
# Full-size configurations in the launch configuration bench.py times: sampled outputs the oracle computes one by one
# (selected pair keys / mesh points are still the exact definition for those outputs), plus identity P4, which holds
# at any size and ties the two kernels together.  The samples are STRATIFIED: besides uniform draws they hold the places
# where a wrong activity-mask bit or a dropped (batch, atom, cubelet) item would live -- whole ragged last batches along
# every axis, the mesh faces (periodic wrap), whole batches of the most crowded regions (most neighbours, most atom
# groups), and pair keys of every kind: on-site, nearest neighbours, pairs at the rim of the cutoff (atoms in different
# groups of a batch, few common cubelets), keys across the cell boundary (R != 0).
def _box_points(w, lo, hi):
    """Flat indices of the mesh points lo <= (i, j, k) < hi (clipped to the mesh)."""
    N = [int(x) for x in w.mesh]
    r = [np.arange(max(0, lo[d]), min(N[d], hi[d]), dtype=np.int64) for d in range(3)]
    return ((r[0][:, None, None] * N[1] + r[1][None, :, None]) * N[2] + r[2][None, None, :]).ravel()


def _stratified_points(w, st, rng, n_uniform):
    from scipy.spatial import cKDTree
    N = np.array([int(x) for x in w.mesh]); bs = np.array([st["batch_bx"], st["batch_by"], st["batch_bz"]]); nb = -(-N // bs)
    parts = [rng.integers(0, w.n_points, n_uniform)]
    # whole last batches along each axis (ragged when bs does not divide N), two per axis
    for ax in range(3):
        for _ in range(2):
            b = rng.integers(0, nb); b[ax] = nb[ax] - 1
            parts.append(_box_points(w, b * bs, (b + 1) * bs))
    # the six mesh faces
    for ax in range(3):
        for side in (0, N[ax] - 1):
            ijk = np.stack([rng.integers(0, N[d], 1500) for d in range(3)], axis=1); ijk[:, ax] = side
            parts.append((ijk[:, 0] * N[1] + ijk[:, 1]) * N[2] + ijk[:, 2])
    # whole batches of the most crowded regions: most atom images within rc + half the batch diagonal of the batch centre
    step = w.cell / N[:, None]
    img = np.concatenate([w.atom_pos + np.array(n) @ w.cell for n in np.ndindex(3, 3, 3)]) - np.array([1, 1, 1]) @ w.cell
    tree = cKDTree(img)
    cand = np.stack([rng.integers(0, nb[d], 4000) for d in range(3)], axis=1)
    centres = ((cand + 0.5) * bs) @ step
    reach = float(w.basis.rcut.max()) + 0.5 * float(np.linalg.norm(bs @ step))
    cnt = np.array([len(x) for x in tree.query_ball_point(centres, reach)])
    for b in cand[np.argsort(-cnt)[:2]]:
        parts.append(_box_points(w, b * bs, (b + 1) * bs))
    return np.unique(np.concatenate(parts)).astype(np.int64)


def _stratified_keys(w, plist, rng, n_uniform):
    A, B, R, off = plist
    d = np.linalg.norm(w.atom_pos[B] + R @ w.cell - w.atom_pos[A], axis=1)
    rim = w.basis.rcut[w.atom_species[A]] + w.basis.rcut[w.atom_species[B]]
    strata = [np.flatnonzero((A == B) & (np.abs(R).sum(1) == 0)),          # on-site
              np.flatnonzero((d > 0) & (d < 3.0)),                             # nearest neighbours
              np.flatnonzero(d > 0.9 * rim),                                   # rim of the cutoff
              np.flatnonzero((d > 0.45 * rim) & (d < 0.55 * rim)),             # middle
              np.flatnonzero(np.abs(R).sum(1) != 0)]                           # across the cell boundary
    parts = [rng.integers(0, len(A), n_uniform)]
    for s in strata:
        if len(s):
            parts.append(rng.choice(s, size=min(len(s), max(8, n_uniform // 5)), replace=False))
    return np.unique(np.concatenate(parts)).astype(np.int64)


def _sampled_parity(torch, cfg, n_keys, n_pts, flag_sets=(0,), seed_extra=None):
    """One oracle evaluation, compared with the library run once per entry of flag_sets (gint_init flags: the default batch shape,
    GINT_FLAG_TUNE as bench.py passes it, a forced shape).  The sampled mesh points are the union of the stratified samples of every
    batch shape that ran.  seed_extra: break the symmetry of D (reading R9: no symmetry assumed)."""
    w = W.make_workload(cfg)
    plist = O.pairs(w)
    V = W.make_potential(w)
    D = W.make_density_blocks(w, *plist)
    if seed_extra is not None:
        D = D + 0.3 * np.random.default_rng(seed_extra).standard_normal(D.size)
    A, B, R, off = plist
    rng = np.random.default_rng([2409, 9399, cfg, 77])
    keys = _stratified_keys(w, plist, rng, n_keys)
    assert len(keys) >= n_keys // 2
    assert np.any(np.abs(R[keys]).sum(1) != 0) or not np.any(np.abs(R).sum(1) != 0)
    dV = abs(np.linalg.det(w.cell)) / w.n_points
    E = _onsite_overlap_closed_form(w) if w.basis.n_species == 1 else None
    onsite = np.flatnonzero((A == B) & (np.abs(R).sum(1) == 0))
    runs, pts_parts = [], []
    for flags in flag_sets:
        g = _gint(w, flags)
        _check_pairs(g, plist)
        st = g.stats()
        st["n_pairs"] = len(A)                      # the oracle's list, just checked key by key against the library's
        pts_parts.append(_stratified_points(w, st, rng, n_pts))
        V_d, D_d = torch.from_numpy(V).cuda(), torch.from_numpy(D).cuda()
        H_d, rho_d = g.vlocal(V_d), g.rho(D_d)
        lhs = float((V_d * rho_d).sum().item() * dV); rhs = float((D_d * H_d).sum().item())
        Hmax, rmax = float(H_d.abs().max().item()), float(rho_d.abs().max().item())
        # run-to-run: accumulation into H and rho is by floating-point atomics (order not fixed): equal to rounding, not bitwise
        H2, rho2 = g.vlocal(V_d), g.rho(D_d)
        rep_H = float((H2 - H_d).abs().max().item()) / Hmax; rep_r = float((rho2 - rho_d).abs().max().item()) / rmax
        del H2, rho2
        # a pin that does not go through the oracle: V == 1 gives the overlap matrix, whose on-site blocks have a closed form
        S = g.vlocal(torch.ones_like(V_d)).cpu().numpy()
        g.close()
        eS = 0.0
        if E is not None:
            eS = max(float(np.max(np.abs(S[off[k]:off[k + 1]].reshape(E.shape) - E))) for k in onsite)
        else:       # several species: orthonormality of every on-site block (real harmonics, normalised radial functions of one l differ)
            no = np.asarray(w.basis.norb)[w.atom_species]
            for k in onsite[::37]:
                blk = S[off[k]:off[k + 1]].reshape(no[A[k]], no[A[k]])
                eS = max(eS, float(np.max(np.abs(np.diag(blk) - 1.0))), float(np.max(np.abs(blk - blk.T))))
        del S
        tag = f"cfg{cfg} flags={flags:#x} batch {st['batch_bx']}x{st['batch_by']}x{st['batch_bz']}"
        assert abs(lhs - rhs) <= 1e-11 * abs(lhs), f"{tag} identity P4 {abs(lhs - rhs) / abs(lhs):.3e}"
        assert rep_H <= 1e-13 and rep_r <= 1e-13, f"{tag} repeatability {rep_H:.3e} {rep_r:.3e}"
        assert eS <= 1e-8, f"{tag} on-site overlap blocks against the closed form {eS:.3e}"
        # keep only the sampled outputs on the host: the H blocks of `keys` and (below) rho at the union of the sampled points
        runs.append((tag, st, [H_d[off[k]:off[k + 1]].cpu().numpy() for k in keys], rho_d.cpu().numpy(), Hmax, rmax))
        del H_d, rho_d, V_d, D_d
        torch.cuda.empty_cache()
    pts = np.unique(np.concatenate(pts_parts)).astype(np.int64)
    assert len(pts) >= n_pts // 2
    H_or = O.vlocal(w, V, plist, sel=keys)
    rho_or = O.rho(w, D, plist, sel=pts)
    for tag, st, Hk, rho, Hmax, rmax in runs:
        # the scale of the tolerance is the largest |H| (|rho|) of the whole result, as in north_star
        eH = max(float(np.max(np.abs(h - H_or[off[k]:off[k + 1]]))) for h, k in zip(Hk, keys)) / Hmax
        er = float(np.max(np.abs(rho[pts] - rho_or[pts]))) / rmax
        assert eH <= TOL, f"{tag} H parity on {len(keys)} sampled keys {eH:.3e}"
        assert er <= TOL, f"{tag} rho parity on {len(pts)} sampled points {er:.3e}"
    return [r[1] for r in runs]


def _onsite_overlap_closed_form(w):
    """S_(A,A,0) = delta_ll' delta_mm' int R_s R_s' r^2 dr for the one-species 2s2p1d basis of the five configs (reading R6:
    r^l exp(-alpha r^2) (1 - (r/rc)^2)^3, normalised), by adaptive quadrature.  rc = 7: 0.859485228247 (s), 0.815140222328 (p)."""
    from scipy.integrate import quad
    rc = float(w.basis.rcut[0])
    alpha = {0: (0.60, 0.20), 1: (0.50, 0.18)}

    def f(r, l, a, b):
        return r ** (2 * l + 2) * np.exp(-(a + b) * r * r) * (1 - (r / rc) ** 2) ** 6

    E = np.eye(13)
    for l, (a1, a2) in alpha.items():
        n1 = quad(f, 0, rc, args=(l, a1, a1), epsabs=1e-15, epsrel=1e-13)[0]
        n2 = quad(f, 0, rc, args=(l, a2, a2), epsabs=1e-15, epsrel=1e-13)[0]
        v = quad(f, 0, rc, args=(l, a1, a2), epsabs=1e-15, epsrel=1e-13)[0] / np.sqrt(n1 * n2)
        if l == 0:
            E[0, 1] = E[1, 0] = v
        else:
            for m in range(3):
                E[2 + m, 5 + m] = E[5 + m, 2 + m] = v
    return E


def test_cfg2_bulk_sampled(torch_cuda):
    """512-atom bulk diamond: up to 7 atom groups per batch (28 tiles), the largest dense contractions."""
    _sampled_parity(torch_cuda, 2, 400, 20000)


def test_cfg3_tbg_sampled(torch_cuda):
    """Default batch shape, and GINT_FLAG_TUNE as bench.py initialises (whatever shape the tuner then keeps)."""
    from paper_2409_09399_b200.gint import FLAG_TUNE
    _sampled_parity(torch_cuda, 3, 600, 50000, flag_sets=(0, FLAG_TUNE))


def test_cfg3_tbg_sampled_nonsymmetric_D(torch_cuda):
    """Full size with a D that has no mirror symmetry: Dh = D + mirror^T of k_sym_D must carry every ordered block (reading R9)."""
    _sampled_parity(torch_cuda, 3, 300, 20000, seed_extra=13)


def test_cfg4_tbg_headline_sampled(torch_cuda):
    """The headline workload (10,444 atoms, 1.76e8 points) in the launch configurations bench.py can time: initialised with
    GINT_FLAG_TUNE exactly as bench.py does (the tuner keeps the default 8x8x16 unless another shape is clearly faster), and with
    the 4x8x16 shape forced, the one the round-2 tuner picked and the committed ncu captures pin."""
    from paper_2409_09399_b200.gint import FLAG_TUNE, batch_flag
    sts = _sampled_parity(torch_cuda, 4, 1000, 100000, flag_sets=(FLAG_TUNE, batch_flag(4, 8, 16)))
    assert (sts[0]["batch_bx"], sts[0]["batch_by"], sts[0]["batch_bz"]) in ((8, 8, 16), (8, 8, 8), (4, 8, 16), (4, 4, 16), (4, 4, 8))
    assert sts[0]["n_pairs"] == 1246278                                         # SURVEY.md P9 (oracle_pairs == library list == this count)
    assert sts[0]["tune_us"] > 0 and (sts[1]["batch_bx"], sts[1]["batch_by"], sts[1]["batch_bz"]) == (4, 8, 16)


def test_cfg5_mixed_species_sampled(torch_cuda):
    """Mixed-species bilayer (13 / 8 / 18 orbitals per atom, rc 7 / 8 / 6, three radial tables): SURVEY 8f NEXT-4."""
    _sampled_parity(torch_cuda, 5, 600, 50000)


def test_repeatability_and_two_live_contexts(torch_cuda):
    """Two contexts alive at once on one device (different shared-memory needs: the big-table path leaves the radial table out of
    shared memory), calls interleaved; and the same call twice gives the same result to rounding."""
    torch = torch_cuda
    w0 = W.make_workload(0)
    pl0 = O.pairs(w0)
    g0 = _gint(w0)
    V0 = torch.from_numpy(W.make_potential(w0)).cuda(); D0 = torch.from_numpy(W.make_density_blocks(w0, *pl0)).cuda()
    H_a, r_a = g0.vlocal(V0).clone(), g0.rho(D0).clone()
    bs = [W.make_basis(9.0, shells=((0, 0.5 + 0.1 * k), (0, 0.2), (1, 0.45), (1, 0.2), (2, 0.35))) for k in range(3)]
    basis = W.Basis(3, np.array([5, 5, 5], np.int32), np.concatenate([b.shell_l for b in bs]), np.array([9.0, 9.0, 9.0]), W.DR,
                    np.concatenate([b.n_knot for b in bs]), np.concatenate([b.tab_y for b in bs]), np.concatenate([b.tab_y2 for b in bs]))
    w1 = W.Workload("big-table", 95, np.diag([22.0, 21.0, 20.0]), np.array([24, 24, 24], np.int32), np.array([0, 1, 2], np.int32),
                    np.array([[3.0, 4.0, 5.0], [9.5, 6.0, 8.0], [15.0, 14.0, 12.0]]), basis)
    g1 = _gint(w1)                              # second live context with another kernel configuration
    assert g1.stats()["tab_in_smem"] == 0 and g0.stats()["tab_in_smem"] == 1
    pl1 = O.pairs(w1)
    V1 = np.random.default_rng(5).standard_normal(w1.n_points)
    H1 = g1.vlocal(torch.from_numpy(V1).cuda()).cpu().numpy()
    H_b, r_b = g0.vlocal(V0), g0.rho(D0)        # the first context still works, and repeats itself
    assert float((H_b - H_a).abs().max() / H_a.abs().max()) <= 1e-13
    assert float((r_b - r_a).abs().max() / r_a.abs().max()) <= 1e-13
    assert _rel(H1, O.vlocal(w1, V1, pl1)) <= TOL
    assert _rel(H_b.cpu().numpy(), O.vlocal(w0, V0.cpu().numpy(), pl0)) <= TOL
    g1.close(); g0.close()


def test_many_orbitals_per_atom(torch_cuda):
    """A species with 31 orbitals (3s 3p 2d... here s,s,s,p,p,p,d,d,d + s: 3 + 9 + 15 + ... <= 32) in a dense cell: eight atoms
    exceed the 104 orbitals of a tile group, so gint_init must cut the batch neighbours into more groups than ceil(n / 8), row
    fragments straddle atoms unevenly and groups hold fewer than eight atoms."""
    torch = torch_cuda
    big = W.make_basis(4.5, shells=((0, 0.8), (0, 0.4), (0, 0.2), (1, 0.7), (1, 0.35), (1, 0.2), (2, 0.6), (2, 0.3), (2, 0.2), (0, 0.12)))
    small = W.make_basis(4.0, shells=((0, 0.5), (1, 0.4)))
    assert int(sum(2 * l + 1 for l in big.shell_l)) == 28
    basis = W.Basis(2, np.array([len(big.shell_l), len(small.shell_l)], np.int32), np.concatenate([big.shell_l, small.shell_l]),
                    np.array([4.5, 4.0]), W.DR, np.concatenate([big.n_knot, small.n_knot]),
                    np.concatenate([big.tab_y, small.tab_y]), np.concatenate([big.tab_y2, small.tab_y2]))
    rng = np.random.default_rng(31)
    cell = np.array([[6.0, 0.0, 0.0], [0.5, 5.5, 0.0], [0.0, 0.3, 6.5]])
    pos = rng.uniform(0, 1, (14, 3)) @ cell
    species = np.array([0, 0, 1, 0, 1, 0, 0, 1, 0, 0, 1, 0, 0, 1], np.int32)
    w = W.Workload("many-orbitals", 96, cell, np.array([20, 18, 22], np.int32), species, pos, basis)
    plist = O.pairs(w)
    g = _gint(w)
    _check_pairs(g, plist)
    V = rng.standard_normal(w.n_points)
    D = rng.standard_normal(int(plist[3][-1]))
    H = g.vlocal(torch.from_numpy(V).cuda()).cpu().numpy()
    rho = g.rho(torch.from_numpy(D).cuda()).cpu().numpy()
    g.close()
    assert _rel(H, O.vlocal(w, V, plist)) <= TOL
    assert _rel(rho, O.rho(w, D, plist)) <= TOL


def test_batch_shape_tuner(torch_cuda):
    """GINT_FLAG_TUNE (the paper's online auto-tuning): gint_init times the candidate batch shapes on a slab of the
    mesh, keeps the default unless another shape is clearly faster, reports what it tried -- and the context it returns is exact."""
    from paper_2409_09399_b200.gint import FLAG_TUNE
    st = _full_parity(torch_cuda, W.make_workload(1), flags=FLAG_TUNE)
    from paper_2409_09399_b200.gint import Gint
    g = Gint.from_workload(W.make_workload(1), flags=FLAG_TUNE)
    rep = g.tune_report()
    st = g.stats()
    g.close()
    tried = [r for r in rep if r[3] > 0]
    assert len(rep) >= 3 and len(tried) >= 2 and 0 < st["tune_us"] < 2_000_000          # "no more than two seconds"
    # the rule of include/gint.h: the default shape (first row) stays unless the fastest other shape is more than 2 % faster
    chosen = (st["batch_bx"], st["batch_by"], st["batch_bz"])
    others = [r for r in tried if r is not rep[0]]
    fastest = min(others, key=lambda r: r[3])
    if rep[0][3] > 0 and not fastest[3] < rep[0][3] * (1.0 - 0.02):
        assert chosen == rep[0][:3]
    else:
        assert chosen == fastest[:3]
    # without the flag nothing is tuned
    g = Gint.from_workload(W.make_workload(0))
    assert g.tune_report() == [] and g.stats()["tune_us"] == 0
    g.close()


def test_unsupported_batch_edge(torch_cuda):
    from paper_2409_09399_b200.gint import GintError, batch_flag
    with pytest.raises(GintError, match="batch edge"):
        _gint(W.make_workload(0), flags=batch_flag(9, 8, 8))


def test_table_too_large_for_shared_memory(torch_cuda):
    """Three species with rc = 9 (901 knots x 5 shells each): the radial table (216 KB) does not fit beside the tile in shared
    memory, so the evaluation reads it from global memory -- the other table path of the kernels."""
    torch = torch_cuda
    bs = [W.make_basis(9.0, shells=((0, 0.5 + 0.1 * k), (0, 0.2), (1, 0.45), (1, 0.2), (2, 0.35))) for k in range(3)]
    basis = W.Basis(3, np.array([5, 5, 5], np.int32), np.concatenate([b.shell_l for b in bs]), np.array([9.0, 9.0, 9.0]), W.DR,
                    np.concatenate([b.n_knot for b in bs]), np.concatenate([b.tab_y for b in bs]), np.concatenate([b.tab_y2 for b in bs]))
    cell = np.diag([22.0, 21.0, 20.0])
    pos = np.array([[3.0, 4.0, 5.0], [9.5, 6.0, 8.0], [15.0, 14.0, 12.0], [6.0, 16.0, 3.0], [11.0, 11.0, 17.0]])
    w = W.Workload("big-table", 93, cell, np.array([40, 38, 36], np.int32), np.array([0, 1, 2, 1, 0], np.int32), pos, basis)
    plist = O.pairs(w)
    g = _gint(w)
    _check_pairs(g, plist)
    rng = np.random.default_rng(21)
    V = rng.standard_normal(w.n_points)
    D = rng.standard_normal(int(plist[3][-1]))
    H = g.vlocal(torch.from_numpy(V).cuda()).cpu().numpy()
    rho = g.rho(torch.from_numpy(D).cuda()).cpu().numpy()
    st = g.stats()
    g.close()
    assert st["tab_in_smem"] == 0                 # the table was left out of shared memory
    assert _rel(H, O.vlocal(w, V, plist)) <= TOL
    assert _rel(rho, O.rho(w, D, plist)) <= TOL


def test_dense_cell_falls_back_to_smaller_batches(torch_cuda):
    """Tiny diamond cell with rc = 8.5 > a: more than 96 atom images touch an 8x8x8 batch, so gint_init must choose a smaller
    batch shape by itself (flags = 0) and still be exact."""
    torch = torch_cuda
    w0 = W.make_workload(0)
    w = W.Workload("dense", 94, w0.cell, np.array([16, 16, 16], np.int32), w0.atom_species, w0.atom_pos, W.make_basis(8.5))
    plist = O.pairs(w)
    g = _gint(w)
    _check_pairs(g, plist)
    st = g.stats()
    assert st["batch_bx"] * st["batch_by"] * st["batch_bz"] < 512 and st["max_nb"] <= 96
    rng = np.random.default_rng(22)
    V = rng.standard_normal(w.n_points)
    D = rng.standard_normal(int(plist[3][-1]))
    H = g.vlocal(torch.from_numpy(V).cuda()).cpu().numpy()
    rho = g.rho(torch.from_numpy(D).cuda()).cpu().numpy()
    g.close()
    assert _rel(H, O.vlocal(w, V, plist)) <= TOL
    assert _rel(rho, O.rho(w, D, plist)) <= TOL
