"""Directed GPU-vs-oracle cases for the kernel paths added in round 2:

* the extra node of a particle that crosses ONE cell face in y or z (k_deposit_mma / k_deposit_tile take it in
  line; crossings in y AND z, and drifts beyond the x window, still go to the per-particle pass) — every
  direction, at tile faces and through the periodic seam, orders 1-3, both precisions;
* the TMA staging of the E/B box against the element-wise cp.async staging: same bits (north_star: "TMA where
  the box is regular"), including tiles smaller than the box (out-of-range parts arrive as zeros) and grids
  whose extents rule TMA out (silent fall-back);
* the drifted-particle list of k_push_tile overflowing (a tile re-walk instead of an in-line gather);
* the fp32 order-1 deposit through the tile's J box in shared memory (k_deposit_smem_cic): small tiles, truncated
  axes, two species, through a re-sort.
"""
import numpy as np
import pytest

import workloads as W
from helpers import compare_state

pytestmark = pytest.mark.gpu

TOL64 = 1e-12
TOL32 = 1e-5


def _pair(n_cells, dx, order, dtype, parts, periodic=(1, 1, 1), tile=(8, 8, 8), gpu_kwargs=None, fields_seed=5,
          sort_interval=4):
    """Oracle and CUDA simulation with the given particles (dict of arrays) and random smooth fields."""
    import oracle
    import paper_2101_12149_b200 as pic
    dt = 0.99 / (W.C_LIGHT * np.sqrt(sum(1.0 / d ** 2 for d in dx)))
    kw = dict(periodic=periodic, tile=tile, sort_interval=sort_interval)
    o = oracle.Oracle(n_cells, dx, dt, order, dtype=dtype, **kw)
    g = pic.Sim(n_cells, dx, dt, order, dtype=dtype, **kw, **(gpu_kwargs or {}))
    a = [np.ascontiguousarray(parts[k], dtype=dtype) for k in ("x", "y", "z", "ux", "uy", "uz", "w")]
    o.add_species(*a, -W.Q_E, W.M_E)
    g.add_species(*a, -W.Q_E, W.M_E)
    rng = np.random.default_rng(fields_seed)
    shape = (n_cells[2], n_cells[1], n_cells[0])
    E = [(1e9 * rng.standard_normal(shape)).astype(dtype) for _ in range(3)]
    B = [(1.0 * rng.standard_normal(shape)).astype(dtype) for _ in range(3)]
    o.set_fields(E, B)
    g.set_fields(E, B)
    return o, g, dt


def _crossers(n_cells, dx, dt, rng, per_case=40):
    """Particles that sit close to a cell face and move across it during ONE step, in every combination of
    {stay, up, down} per axis (27 cases), in cells spread over the grid including the tile faces and the
    periodic seam. |u| is chosen so that the move is 0.05-0.2 cell: across the near face, never two."""
    xs = {k: [] for k in ("x", "y", "z", "ux", "uy", "uz", "w")}
    n = np.asarray(n_cells)
    for cx in (-1, 0, 1):
        for cy in (-1, 0, 1):
            for cz in (-1, 0, 1):
                cell = np.stack([rng.integers(0, n[d], per_case) for d in range(3)], axis=1)
                # a third of the cells on tile faces / the seam: 0, 7, 8, N-1
                pick = rng.random((per_case, 3)) < 0.35
                special = np.stack([rng.choice([0, 7 % n[d], 8 % n[d], n[d] - 1], per_case) for d in range(3)], axis=1)
                cell = np.where(pick, special, cell)
                frac = np.empty((per_case, 3))
                vel = np.empty((per_case, 3))
                for d, c in enumerate((cx, cy, cz)):
                    move = rng.uniform(0.05, 0.2, per_case)          # cells per step along this axis
                    if c == 0:
                        frac[:, d] = rng.uniform(0.35, 0.65, per_case)
                        vel[:, d] = rng.choice([-1.0, 1.0], per_case) * rng.uniform(0.0, 0.15, per_case)
                    elif c > 0:
                        frac[:, d] = 1.0 - rng.uniform(0.0, 0.9, per_case) * move
                        vel[:, d] = move
                    else:
                        frac[:, d] = rng.uniform(0.0, 0.9, per_case) * move
                        vel[:, d] = -move
                pos = (cell + np.clip(frac, 1e-9, 1 - 1e-9)) * np.asarray(dx)
                v = vel * np.asarray(dx) / dt                       # m/s, |v| < c by the CFL bound
                beta2 = np.sum(v ** 2, axis=1) / W.C_LIGHT ** 2
                assert np.all(beta2 < 0.9)
                gamma = 1.0 / np.sqrt(1.0 - beta2)
                u = v * gamma[:, None]
                for d, k in enumerate("xyz"):
                    xs[k].append(pos[:, d])
                    xs["u" + k].append(u[:, d])
                xs["w"].append(rng.uniform(0.5, 1.5, per_case) * 1e6)
    return {k: np.concatenate(v) for k, v in xs.items()}


@pytest.mark.parametrize("order", [1, 2, 3])
@pytest.mark.parametrize("dtype,mode", [(np.float64, 0), (np.float64, 3), (np.float32, 0), (np.float32, 4)])
def test_face_crossings_in_every_direction_match_the_oracle(order, dtype, mode):
    """One step from identical state with particles built to cross cell faces in all 27 direction
    combinations. Weak fields (the push must not turn the particles around): what is tested is the deposit.
    J is compared element by element; the crossing statistics are asserted so that every path is really hit."""
    n_cells, dx = (24, 16, 16), (1.0e-6, 0.8e-6, 0.6e-6)
    rng = np.random.default_rng(1234 + order)
    dt = 0.99 / (W.C_LIGHT * np.sqrt(sum(1.0 / d ** 2 for d in dx)))
    parts = _crossers(n_cells, dx, dt, rng)
    o, g, _ = _pair(n_cells, dx, order, dtype, parts, gpu_kwargs=dict(deposit_mode=mode))
    zero = [np.zeros((n_cells[2], n_cells[1], n_cells[0]), dtype=dtype) for _ in range(3)]
    o.set_fields(zero, zero)
    g.set_fields(zero, zero)
    g.sort_now()
    o.sort_now()
    before = o.get_particles(0)
    o.step(1)
    g.step(1)
    tol = TOL64 if dtype == np.float64 else TOL32
    errs = compare_state(o, g, tol)
    after = o.get_particles(0)
    # the sort at step 0 is the identity now, so slots correspond
    assert np.array_equal(before["id"], after["id"])
    moved = []
    for d, k in enumerate("xyz"):
        L = n_cells[d] * dx[d]
        c0 = np.floor(before[k] / dx[d]).astype(int)
        c1 = np.floor(after[k] / dx[d]).astype(int)
        dc = (c1 - c0 + n_cells[d] // 2) % n_cells[d] - n_cells[d] // 2      # through the seam: +-1
        moved.append(dc)
        assert np.all(np.abs(dc) <= 1)
        assert np.all((after[k] >= 0) & (after[k] < L))
    moved = np.stack(moved, axis=1)
    for ax in (1, 2):
        assert np.sum(moved[:, ax] == 1) > 100 and np.sum(moved[:, ax] == -1) > 100       # single crossings
    assert np.sum((moved[:, 1] != 0) & (moved[:, 2] != 0)) > 100                          # y and z at once
    assert np.sum((moved[:, 0] != 0) & (moved[:, 1] != 0) & (moved[:, 2] == 0)) > 50      # x and y
    assert errs["J"] <= tol


@pytest.mark.parametrize("order", [1, 2, 3])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n_cells,tile", [((24, 16, 16), (8, 8, 8)), ((12, 12, 12), (4, 4, 4)), ((16, 8, 24), (8, 4, 8))])
def test_tma_staging_gives_the_same_bits_as_cp_async(order, dtype, n_cells, tile):
    """pic_options.box_staging: the box brought by one TMA tensor copy (x fastest, 12 x 14 x 12, starting two
    nodes below the tile) and the box copied element by element (y fastest, padded x stride) hold the same
    values, so particles and fields agree bit for bit after several steps (deterministic deposition makes J
    exact too). Tiles of 4 cells: the box reaches past the padded array and TMA fills zeros there."""
    import paper_2101_12149_b200 as pic
    cfg = W.scaled(W.CONFIGS["C2"], n_cells, tile=tile, dx=(1.0e-6, 0.9e-6, 0.7e-6))
    cfg.order = order
    cfg.dtype = "f64" if dtype == np.float64 else "f32"
    cfg.species[0].sigma = 0.2
    species, _, _ = W.generate(cfg)
    E, B = W.random_fields(cfg, np.random.default_rng(3))
    out = []
    for staging in (1, 2):          # PIC_STAGE_CP_ASYNC, PIC_STAGE_TMA
        g = pic.Sim(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, dtype=cfg.np_dtype, tile=tile, sort_interval=4,
                    deterministic=True, box_staging=staging)
        a = [species[0][1][k] for k in ("x", "y", "z", "ux", "uy", "uz", "w")]
        g.add_species(*a, -W.Q_E, W.M_E)
        g.set_fields(E, B)
        g.step(6)
        out.append((g.get_fields(), g.get_particles(0)))
    for grp in range(3):
        for a, b in zip(out[0][0][grp], out[1][0][grp]):
            assert np.array_equal(a, b)
    for k in ("id", "x", "y", "z", "ux", "uy", "uz", "w"):
        assert np.array_equal(out[0][1][k], out[1][1][k]), k


def test_tma_request_falls_back_where_the_strides_rule_it_out():
    """An odd grid (padded extent 15 + 8 = 23 nodes: the y stride is not a multiple of 16 bytes) and an odd
    tile: PIC_STAGE_TMA silently uses cp.async, and the step still matches the oracle."""
    n_cells, dx = (15, 10, 9), (1.0e-6, 0.8e-6, 0.6e-6)
    rng = np.random.default_rng(9)
    npart = 6000
    parts = {k: rng.random(npart) * n_cells[d] * dx[d] for d, k in enumerate("xyz")}
    for k in ("ux", "uy", "uz"):
        parts[k] = 0.05 * W.C_LIGHT * rng.standard_normal(npart)
    parts["w"] = np.full(npart, 1e6)
    o, g, _ = _pair(n_cells, dx, 3, np.float64, parts, tile=(5, 5, 3), gpu_kwargs=dict(box_staging=2))
    o.step(3)
    g.step(3)
    compare_state(o, g, 20 * TOL64)


@pytest.mark.parametrize("staging", [1, 2])
def test_drift_list_overflow_rewalks_the_tile(staging):
    """Very hot particles and a sort only every 8 steps: after a few steps more than 256 particles of a tile
    have left its box, the shared-memory list overflows and the second pass of k_push_tile re-walks the tile.
    The result matches the oracle and is the same from run to run."""
    import paper_2101_12149_b200 as pic
    cfg = W.scaled(W.CONFIGS["C2"], (16, 16, 16), dx=(1.0e-6, 0.9e-6, 0.7e-6))
    cfg.species[0].sigma = 0.6
    cfg.sort_interval = 8
    import oracle
    species, _, _ = W.generate(cfg)
    E, B = W.random_fields(cfg, np.random.default_rng(4))
    a = [species[0][1][k] for k in ("x", "y", "z", "ux", "uy", "uz", "w")]
    o = oracle.Oracle(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, dtype=cfg.np_dtype, tile=cfg.tile, sort_interval=8)
    o.add_species(*a, -W.Q_E, W.M_E)
    o.set_fields(E, B)
    runs = []
    for rep in range(2):
        g = pic.Sim(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, dtype=cfg.np_dtype, tile=cfg.tile, sort_interval=8,
                    deterministic=True, box_staging=staging)
        g.add_species(*a, -W.Q_E, W.M_E)
        g.set_fields(E, B)
        g.step(7)
        runs.append(g)
    o.step(7)
    # how many particles sit outside their sort-time tile's box by now (cell more than 1 below / 2 above the tile)
    po = o.get_particles(0)
    cell, perm = o.get_sort_state(0)
    compare_state(o, runs[0], 50 * TOL64)
    p0, p1 = runs[0].get_particles(0), runs[1].get_particles(0)
    for k in ("id", "x", "y", "z", "ux", "uy", "uz", "w"):
        assert np.array_equal(p0[k], p1[k]), k
    # the premise: at the sort (step 0) every particle is in its tile; 7 steps later a hot plasma has moved
    # > 256 of a tile's 4096 particles more than a cell beyond the tile (0.6 c x 7 steps ~ 1.4 cells rms)
    x_now = np.stack([po[k] / cfg.dx[d] for d, k in enumerate("xyz")], axis=1)
    cz, rem = np.divmod(cell, cfg.n_cells[0] * cfg.n_cells[1])
    cy, cx = np.divmod(rem, cfg.n_cells[0])
    c_sort = np.stack([cx, cy, cz], axis=1)
    tile0 = (c_sort // 8) * 8
    rel = x_now - tile0
    rel = (rel + 4) % np.asarray(cfg.n_cells) - 4          # periodic distance from the tile base, in [-4, N-4)
    out_of_box = np.any((rel < -0.5) | (rel > 9.5), axis=1)
    counts = np.bincount((tile0[:, 0] // 8) + 2 * (tile0[:, 1] // 8) + 4 * (tile0[:, 2] // 8), weights=out_of_box, minlength=8)
    assert counts.max() > 256, counts


@pytest.mark.parametrize("n_cells,tile,periodic", [((16, 16, 16), (8, 8, 8), (1, 1, 1)), ((12, 8, 20), (4, 4, 4), (1, 1, 0)),
                                                   ((24, 8, 8), (8, 4, 8), (0, 1, 1))])
def test_fp32_order1_shared_memory_deposit_matches_the_oracle(n_cells, tile, periodic):
    """k_deposit_smem_cic (AUTO in fp32 at order 1: the tile's J box in shared memory): two species, hot enough
    that particles cross cell and tile faces, tiles smaller than 8 cells, truncated axes (particles leave and
    are deactivated, J deposited outside is dropped), several steps through a re-sort; and the same bits of
    x, u as the lane-group kernel (explicit PIC_DEPOSIT_TILE), which shares nothing but the push with it."""
    import oracle
    import paper_2101_12149_b200 as pic
    cfg = W.scaled(W.CONFIGS["C5"], n_cells, tile=tile, periodic=periodic, dx=(1.0e-6, 0.8e-6, 0.7e-6))
    cfg.order = 1
    cfg.dtype = "f32"
    species, _, _ = W.generate(cfg)
    E, B = W.random_fields(cfg, np.random.default_rng(11))
    kw = dict(periodic=periodic, tile=tile, sort_interval=4)
    o = oracle.Oracle(cfg.n_cells, cfg.dx, cfg.dt, 1, dtype=np.float32, **kw)
    sims = [pic.Sim(cfg.n_cells, cfg.dx, cfg.dt, 1, dtype=np.float32, deposit_mode=m, **kw) for m in (0, 3)]
    for spec, arrs in species:
        a = [arrs[k] for k in ("x", "y", "z", "ux", "uy", "uz", "w")]
        o.add_species(*a, spec.charge, spec.mass)
        for g in sims:
            g.add_species(*a, spec.charge, spec.mass)
    o.set_fields(E, B)
    for g in sims:
        g.set_fields(E, B)
    o.step(1)
    for g in sims:
        g.step(1)
    compare_state(o, sims[0], TOL32, n_species=2)
    o.step(5)
    for g in sims:
        g.step(5)
    compare_state(o, sims[0], 20 * TOL32, n_species=2)
    assert o.diagnostics()["deactivated"] == sims[0].diagnostics()["deactivated"]
    if 0 in periodic:
        assert sims[0].diagnostics()["deactivated"] > 0
    for s in range(2):
        p0, p1 = sims[0].get_particles(s), sims[1].get_particles(s)
        assert np.array_equal(p0["id"], p1["id"])
    J0, J1 = sims[0].get_fields()[2], sims[1].get_fields()[2]
    scale = max(np.max(np.abs(a)) for a in J1)
    assert max(np.max(np.abs(a.astype(np.float64) - b)) for a, b in zip(J0, J1)) <= 20 * TOL32 * scale
