"""sph_prefix_sum_noalloc (include/sph.h): the allocation-free variant of the scan step N6 against the existing path.

Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test.  The existing path is the
scan inside sph_neighbors_export (same kernels, block sums in a context buffer that grows on demand): it turns the
per-row counts of the caller-order lists into the exported row_ptr.  Integer work, so the bar is bit-exact."""
import numpy as np
import pytest
import torch

from paper_2507_21684_b200 import workloads as W
from paper_2507_21684_b200.binding import Sph, SphError, prefix_sum_noalloc, PREFIX_SUM_NOALLOC_MAX

pytestmark = pytest.mark.gpu


def _existing_path(wl):
    """row_ptr of sph_neighbors_export and the counts it was scanned from"""
    sph = Sph(0)
    try:
        dev = "cuda:0"
        sph.build_cells(wl.domain, torch.from_numpy(wl.x).to(dev), torch.from_numpy(wl.h).to(dev))
        sph.neighbors(1.0)
        row_ptr, _ = sph.neighbors_export()
        torch.cuda.synchronize()
        return row_ptr.clone()
    finally:
        sph.close()


def test_prefix_sum_noalloc_matches_the_existing_scan_on_two_calls_in_a_row():
    big = _existing_path(W.perturbed(W.make(3, n_axis=40), amp_x=0.3))       # 64 000 rows: 16 scan tiles, ragged tail
    small = _existing_path(W.perturbed(W.make(1, n_axis=50), amp_x=0.3))     # 2 500 rows: one tile
    prefix_sum_noalloc(torch.empty(0, dtype=torch.int32, device="cuda:0"),
                       torch.empty(1, dtype=torch.int64, device="cuda:0"))    # n = 0: the per-device set-up only
    # two calls in a row on one stream, the larger first: the second finds the first one's block sums in the shared array
    for ref in (big, small, big):
        counts = (ref[1:] - ref[:-1]).to(torch.int32).contiguous()
        out = torch.full((ref.numel(),), -7, dtype=torch.int64, device="cuda:0")
        free_before = torch.cuda.mem_get_info()[0]
        prefix_sum_noalloc(counts, out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before                    # nothing was allocated on the device
        assert torch.equal(out, ref)                                          # bit-exact against the existing path
        assert torch.equal(out[1:], torch.cumsum(counts.to(torch.int64), 0)) and int(out[0]) == 0


def test_prefix_sum_noalloc_large_values_and_size_limit():
    # totals beyond 2^32 (the offsets are 64-bit, as C4's 2.3e9 entries need), n not a multiple of the scan tile
    n = 3 * 4096 + 17
    g = torch.Generator(device="cpu").manual_seed(5)
    c = torch.randint(0, 2 ** 31 - 1, (n,), generator=g, dtype=torch.int64)
    counts = c.to(torch.int32).cuda()
    out = torch.empty(n + 1, dtype=torch.int64, device="cuda:0")
    prefix_sum_noalloc(counts, out)
    ref = np.concatenate([[0], np.cumsum(c.numpy())])
    assert int(ref[-1]) > 2 ** 32 and np.array_equal(out.cpu().numpy(), ref)
    # beyond the stated maximum: rejected with its own error code, nothing launched (the buffers are never touched, so
    # tiny ones stand in for them)
    from paper_2507_21684_b200.binding import load_library, _ptr
    lib = load_library()
    rc = lib.sph_prefix_sum_noalloc(0, _ptr(counts), _ptr(out), PREFIX_SUM_NOALLOC_MAX + 1, None)
    assert rc == -6 and b"capacity" in lib.sph_strerror(rc)
    assert lib.sph_prefix_sum_noalloc(0, None, None, 5, None) == -1
    assert lib.sph_prefix_sum_noalloc(-1, _ptr(counts), _ptr(out), 5, None) == -1
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref)
