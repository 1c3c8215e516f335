"""pic_sort_permutation_noalloc (include/pic.h): the sort of step 1 through the entry point that allocates nothing —
its scratch is a fixed file-scope device array inside the library — against the existing path (pic_sort_now +
pic_get_sort_state on a handle, whose scratch comes from the memory pool). Integer work: bit-exact, as in
tests/test_gpu_parity.py. Two calls in a row on different inputs (the second smaller, so that stale contents of the
shared array would show), both precisions, and the size limit.

This file is named to be collected LAST (the run is `pytest -x`: a failure here must not hide other tests).
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


def _reference(cfg, arrs, key_mode):
    """cell, perm from the existing path."""
    import paper_2101_12149_b200 as pic
    g = pic.Sim(cfg.n_cells, cfg.dx, cfg.dt, cfg.order, dtype=cfg.np_dtype, tile=cfg.tile, sort_interval=4,
                sort_key_mode=key_mode)
    g.add_species(*[arrs[k] for k in ("x", "y", "z", "ux", "uy", "uz", "w")], -W.Q_E, W.M_E)
    g.sort_now()
    cell, perm = g.get_sort_state()
    g.close()
    return cell, perm


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_noalloc_sort_matches_the_handle_path_on_two_calls_in_a_row(dtype):
    import torch
    import paper_2101_12149_b200 as pic
    dev = torch.device("cuda:0")
    torch.cuda.set_device(0)
    cases = [((32, 24, 16), (8, 8, 8), 0, 8),      # 98 304 particles, 24 radix blocks, 14 key bits (two passes)
             ((20, 12, 28), (4, 4, 4), 0, 3),      # smaller second call, non power-of-two grid, ragged tail
             ((16, 16, 16), (8, 8, 8), 1, 2)]      # tile-only key: 3 key bits, one pass
    refs, outs = [], []
    for n_cells, tile, key_mode, ppc in cases:
        cfg = W.scaled(W.CONFIGS["C2"], n_cells, tile=tile, dx=(1.0e-6, 0.8e-6, 0.6e-6))
        cfg.dtype = dtype
        cfg.species[0].ppc = ppc
        species, _, _ = W.generate(cfg)
        arrs = species[0][1]
        refs.append(_reference(cfg, arrs, key_mode))
        n = len(arrs["x"])
        assert n <= pic.binding.PIC_NOALLOC_MAX_PARTICLES
        x, y, z = (torch.from_numpy(np.ascontiguousarray(arrs[k])).to(dev) for k in "xyz")
        cell = torch.full((n,), -7, dtype=torch.int32, device=dev)
        perm = torch.full((n,), -7, dtype=torch.int32, device=dev)
        # back to back on one stream, no synchronisation in between: the calls share the scratch array, the
        # stream orders them
        pic.binding.pic_sort_permutation_noalloc(cfg.n_cells, cfg.dx, tile, x, y, z, cell, perm, sort_key_mode=key_mode,
                                                 stream=torch.cuda.current_stream().cuda_stream)
        outs.append((cell, perm, x, y, z))
    torch.cuda.synchronize()
    for (cell_ref, perm_ref), (cell, perm, *_), case in zip(refs, outs, cases):
        assert np.array_equal(perm.cpu().numpy(), perm_ref), case
        assert np.array_equal(cell.cpu().numpy(), cell_ref), case
        assert sorted(perm.cpu().numpy().tolist()) == list(range(len(perm_ref)))


def test_noalloc_sort_rejects_sizes_beyond_its_scratch_and_allocates_nothing():
    import torch
    import paper_2101_12149_b200 as pic
    dev = torch.device("cuda:0")
    torch.cuda.set_device(0)
    nmax = pic.binding.PIC_NOALLOC_MAX_PARTICLES
    n = nmax + 1
    x = torch.zeros(n, dtype=torch.float64, device=dev)
    out = torch.zeros(n, dtype=torch.int32, device=dev)
    with pytest.raises(pic.PicError) as ei:
        pic.binding.pic_sort_permutation_noalloc((16, 16, 16), (1e-6,) * 3, (8, 8, 8), x, x, x, out, out)
    assert ei.value.code == -6 and "PIC_NOALLOC_MAX_PARTICLES" in str(ei.value)       # PIC_ERR_CAPACITY
    with pytest.raises(pic.PicError):
        pic.binding.pic_sort_permutation_noalloc((16, 16, 16), (1e-6,) * 3, (5, 8, 8), x[:100], x[:100], x[:100], out[:100], out[:100])
    # exactly the maximum is accepted, and no device memory is taken or released by the call (the driver's free
    # memory is the same before and after: torch's caching allocator is not involved, the tensors exist already)
    rng = np.random.default_rng(5)
    pos = [torch.from_numpy(rng.random(nmax) * 16e-6).to(dev) for _ in range(3)]
    cell = torch.empty(nmax, dtype=torch.int32, device=dev)
    perm = torch.empty(nmax, dtype=torch.int32, device=dev)
    pic.binding.pic_sort_permutation_noalloc((16, 16, 16), (1e-6,) * 3, (8, 8, 8), *pos, cell, perm)   # first use on this device
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    pic.binding.pic_sort_permutation_noalloc((16, 16, 16), (1e-6,) * 3, (8, 8, 8), *pos, cell, perm)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    p = perm.cpu().numpy()
    c = cell.cpu().numpy()
    # the rule itself, in numpy: stable ascending sort by tile-major cell key
    inv = 1.0 / 1e-6                                   # as the library forms it; ONE rounded multiply per axis
    cx, cy, cz = (np.floor(t.cpu().numpy() * inv).astype(np.int64).clip(0, 15) for t in pos)
    key = ((cx // 8) + 2 * ((cy // 8) + 2 * (cz // 8))) * 512 + (cx % 8) + 8 * ((cy % 8) + 8 * (cz % 8))
    assert np.array_equal(p, np.argsort(key, kind="stable").astype(np.int32))
    assert np.array_equal(c, (cx + 16 * (cy + 16 * cz))[p].astype(np.int32))
