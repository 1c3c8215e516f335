"""Shared by the GPU parity tests: build the oracle and the CUDA simulation from the same seeded
inputs (workloads module) and compare array families with the normalisation BASELINE.json states."""
import numpy as np

import workloads as W


def make_pair(cfg, fields="config", shuffle=True, gpu_kwargs=None, with_oracle=True, rng_fields_seed=77,
              method=None):
    """(oracle or None, gpu Sim, species arrays) for a workloads.Config."""
    import oracle
    import paper_2101_12149_b200 as pic
    species, E, B = W.generate(cfg, shuffle=shuffle)
    if fields == "random":
        E, B = W.random_fields(cfg, np.random.default_rng(rng_fields_seed))
    kw = dict(periodic=cfg.periodic, tile=cfg.tile, sort_interval=cfg.sort_interval)
    kw.update(method or {})          # pusher= / gather_mode= / solver=, same values on both sides
    o = None
    if with_oracle:
        o = oracle.Oracle(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, dtype=cfg.np_dtype, **kw)
    g = pic.Sim(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, dtype=cfg.np_dtype, **kw, **(gpu_kwargs or {}))
    for spec, arrs in species:
        a = [arrs[k] for k in ("x", "y", "z", "ux", "uy", "uz", "w")]
        if o is not None:
            o.add_species(*a, spec.charge, spec.mass)
        g.add_species(*a, spec.charge, spec.mass)
    if E is not None:
        if o is not None:
            o.set_fields(E, B)
        g.set_fields(E, B)
    return o, g, species


def family_err(a_list, b_list):
    """max |a-b| over a family of arrays, normalised by the family's max |value| (north_star)."""
    scale = max(float(np.max(np.abs(np.asarray(b, dtype=np.float64)))) if np.size(b) else 0.0 for b in b_list)
    err = max(float(np.max(np.abs(np.asarray(a, dtype=np.float64) - np.asarray(b, dtype=np.float64)))) if np.size(b) else 0.0
              for a, b in zip(a_list, b_list))
    return err / scale if scale > 0 else err


def compare_state(o, g, tol, n_species=1, check_J=True):
    """One-step comparison from identical state: particles (same order) and E, B, J."""
    out = {}
    Eo, Bo, Jo = o.get_fields()
    Eg, Bg, Jg = g.get_fields()
    out["E"] = family_err(Eg, Eo)
    out["B"] = family_err(Bg, Bo)
    if check_J:
        out["J"] = family_err(Jg, Jo)
    for s in range(n_species):
        po, pg = o.get_particles(s), g.get_particles(s)
        assert np.array_equal(po["id"], pg["id"]), "particle order differs"
        out["x%d" % s] = family_err([pg[k] for k in "xyz"], [po[k] for k in "xyz"])
        out["u%d" % s] = family_err([pg[k] for k in ("ux", "uy", "uz")], [po[k] for k in ("ux", "uy", "uz")])
        out["w%d" % s] = family_err([pg["w"]], [po["w"]])
    bad = {k: v for k, v in out.items() if not (v <= tol)}
    assert not bad, "beyond tolerance %g: %s (all: %s)" % (tol, bad, out)
    return out
