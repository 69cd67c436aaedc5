"""hair_scan_noalloc against the frame's own scan.

Why the entry point exists: some users of libhair cannot let it allocate device memory — a renderer whose own pool
took all of the GPU's memory at start-up (a cudaMalloc in its frame loop fails or stalls the device), or a host that
bans the synchronising cudaMalloc / cudaFree from its per-frame code. Everything else in the library works through a
context that allocates its scratch; hair_scan_noalloc takes the caller's buffers only and keeps its tile sums in a fixed
array in the library's device code (at most binding.SCAN_NOALLOC_MAX bundle-instances, shared by all calls).

What is checked: on the bundle tables of two different frames, one call after the other with no reset in between (the
array keeps the first call's sums), the scans equal columns .z / .w of the table that k_lod + k_scan wrote and the
totals equal hair_stats — bit for bit, the bar of every integer stage in tests/test_gpu_parity.py. The second and third
calls are shorter than the first, so a stale sum of the longer call would show.

This file sorts last on purpose (pytest -x stops at the first failure); it must pass alone and after the others.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2607_04230_b200 import binding, synth


def test_size_beyond_the_fixed_array_is_refused_before_any_cuda_call():
    """No GPU needed: the size check comes first and names the limit (pointers are never touched)."""
    L = binding.load()
    fake = C.c_void_p(0x1000)
    rc = L.hair_scan_noalloc(0, None, fake, binding.SCAN_NOALLOC_MAX + 1, fake, fake)
    assert rc == -1  # HAIR_E_INVALID_ARG
    msg = L.hair_scan_noalloc_error().decode()
    assert str(binding.SCAN_NOALLOC_MAX) in msg and "HAIR_SCAN_NOALLOC_MAX" in msg, msg
    assert L.hair_scan_noalloc(0, None, C.c_void_p(0x1004), 8, fake, fake) == -1  # misaligned
    assert "aligned" in L.hair_scan_noalloc_error().decode()
    assert L.hair_scan_noalloc(0, None, fake, 8, fake, None) == -1  # no totals
    assert "null" in L.hair_scan_noalloc_error().decode()


def _frame_table(h, sc, lam):
    import torch
    h.render(sc["camera"], lam)
    torch.cuda.synchronize()
    st = h.stats()
    return h.debug_table(), st  # int32 [n_bi][4] = {N_LOD, C, slot_base, vertex_base} (a copy)


def _check(table, n, n_strands, n_vertices):
    """Scan the first n rows through the no-alloc call; the existing path's scan of a prefix is the prefix of its scan."""
    import torch
    counts = table[:n, 0:2].contiguous()
    bases = torch.full((n, 2), -1, dtype=torch.int32, device=table.device)
    totals = torch.full((2,), -1, dtype=torch.int32, device=table.device)
    binding.scan_noalloc(counts, bases, totals)
    torch.cuda.synchronize()
    assert torch.equal(bases, table[:n, 2:4]), "slot_base / vertex_base differ from k_scan's"
    assert totals.cpu().numpy().view(np.uint32).tolist() == [n_strands, n_vertices]


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_frame_scan():
    import torch
    sc = synth.config(4, scale=0.05, res_scale=0.25)  # five grooms, 64 tiles of 256 bundle-instances
    h = binding.Hair(0)
    for g in sc["grooms"]:
        h.mesh_upload(g)
    h.set_render_params(sc["params"])
    # call 1: the frame with the config's own per-groom lambda (LOD thins the far grooms, some bundles culled)
    t1, s1 = _frame_table(h, sc, sc["lam"])
    n_bi = t1.shape[0]
    assert n_bi == s1["n_bundles"] and n_bi > 3 * 256
    assert 0 < s1["n_strands_lod"] < s1["n_strands_total"]
    _check(t1, n_bi, s1["n_strands_lod"], s1["n_vertices"])
    # call 2, straight after: another frame (LOD off: every count differs), scanned over a ragged prefix that ends
    # inside a tile. Its totals are the bases of the first row left out.
    t2, s2 = _frame_table(h, sc, [0.0])
    assert s2["n_strands_lod"] == s2["n_strands_total"] and not torch.equal(t1, t2)
    n2 = 2 * 256 + 77
    exp = t2[n2, 2:4].cpu().numpy().view(np.uint32).tolist()
    _check(t2, n2, exp[0], exp[1])
    # and the whole of it, one tile or less, nothing
    _check(t2, n_bi, s2["n_strands_lod"], s2["n_vertices"])
    _check(t2, 200, *t2[200, 2:4].cpu().numpy().view(np.uint32).tolist())
    _check(t2, 0, 0, 0)
    h.close()


@pytest.mark.gpu
def test_maximum_size_runs_and_one_more_is_refused():
    import torch
    n = binding.SCAN_NOALLOC_MAX
    gen = torch.Generator(device="cuda").manual_seed(7)
    counts = torch.stack([torch.randint(0, 40, (n,), generator=gen, device="cuda", dtype=torch.int32),
                          torch.randint(3, 100, (n,), generator=gen, device="cuda", dtype=torch.int32)], dim=1).contiguous()
    bases = torch.empty_like(counts)
    totals = torch.empty(2, dtype=torch.int32, device="cuda")
    binding.scan_noalloc(counts, bases, totals)
    torch.cuda.synchronize()
    s = counts[:, 0].to(torch.int64)
    v = s * counts[:, 1].to(torch.int64)
    # sums stay below 2^32 here (40 * 100 * 2^20 < 2^32): compare as unsigned
    u = lambda x: x.to(torch.int64) & 0xFFFFFFFF
    assert torch.equal(u(bases[:, 0]), torch.cumsum(s, 0) - s) and torch.equal(u(bases[:, 1]), torch.cumsum(v, 0) - v)
    assert [int(x) for x in u(totals)] == [int(s.sum()), int(v.sum())]
    big = torch.empty((n + 1, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(binding.HairError, match="HAIR_SCAN_NOALLOC_MAX"):
        binding.scan_noalloc(big, big, totals)
