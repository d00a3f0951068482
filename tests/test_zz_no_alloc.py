"""bbtn_region_bound_static: the K5 region bound with its scratch in a file-scope device array (no device
allocation), against the ordinary bbtn_region_bound on the same inputs.  Integer work: bit-exact.
Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2602_05470_b200 import instances as I

pytestmark = pytest.mark.gpu

MAX_ITEMS = 1 << 20


def _grid_regions(rows, cols, br, bc, ids=None):
    offs, verts = [0], []
    for r0 in range(0, rows, br):
        for c0 in range(0, cols, bc):
            for r in range(r0, min(r0 + br, rows)):
                for c in range(c0, min(c0 + bc, cols)):
                    v = r * cols + c if ids is None else ids[r][c]
                    if v >= 0:
                        verts.append(v)
            offs.append(len(verts))
    return np.array(offs, np.int32), np.array(verts, np.int32)


@pytest.mark.parametrize("kind", ["ising", "king"])
def test_region_bound_static_equals_region_bound_two_calls_in_a_row(kind):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2602_05470_b200 import binding as bb
    bb.load()
    rows, cols = 9, 10
    if kind == "ising":
        inst = I.ising_lattice_2d(rows, cols, 5, field_h=1)
        ids = None
    else:
        inst = I.kings_subgraph(rows, cols, 0.8, 7, weights="rand")
        ids = -np.ones((rows, cols), int); ids[inst.meta["keep"]] = np.arange(inst.n_vertices)
    offs, verts = _grid_regions(rows, cols, 3, 3, ids)
    f = 9
    fixed = I.random_order(inst.n_vertices, 31)[:f]
    assign = I.all_assignments(f)                                   # 512 leaves x 12 regions
    h = bb.Handle(inst)                                             # host-pointer handle: the static call takes device pointers anyway
    want = h.region_bound(offs, verts, fixed, assign)               # the existing path; also caches the K5 tables (set-up)
    h.region_bound_static(offs, verts, fixed, None, None, B=0)      # set-up call: resolves the array's address, launches nothing

    a1 = torch.from_numpy(assign).cuda()
    out1 = torch.full((len(assign),), 12345, dtype=torch.int32, device="cuda")
    # second call: fewer leaves, other rows -- the array still holds the first call's maxima
    rows2 = np.ascontiguousarray(assign[::-1][:200])
    a2 = torch.from_numpy(rows2).cuda()
    out2 = torch.full((200,), 12345, dtype=torch.int32, device="cuda")
    free_before = torch.cuda.mem_get_info()[0]
    h.region_bound_static(offs, verts, fixed, a1, out1)
    h.region_bound_static(offs, verts, fixed, a2, out2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before              # nothing was allocated on the device
    assert np.array_equal(out1.cpu().numpy(), want)
    assert np.array_equal(out2.cpu().numpy(), want[::-1][:200])
    # and once more after the other size, on a non-default stream
    s = torch.cuda.Stream()
    out3 = torch.zeros(len(assign), dtype=torch.int32, device="cuda")
    s.wait_stream(torch.cuda.current_stream())
    h.region_bound_static(offs, verts, fixed, a1, out3, stream=s.cuda_stream)
    s.synchronize()
    assert np.array_equal(out3.cpu().numpy(), want)

    # no regions: the sum kernel alone (reads nothing from the array)
    want0 = h.region_bound([0], [], fixed, assign)
    out0 = torch.zeros(len(assign), dtype=torch.int32, device="cuda")
    h.region_bound_static([0], [], fixed, a1, out0)
    torch.cuda.synchronize()
    assert np.array_equal(out0.cpu().numpy(), want0)

    # beyond the static maximum: refused, clearly
    n_reg = len(offs) - 1
    too_many = MAX_ITEMS // n_reg + 1
    with pytest.raises(bb.BbtnError) as ei:
        h.region_bound_static(offs, verts, fixed, a1, out1, B=too_many)
    assert ei.value.status == bb.BBTN_ESHAPE and "exceeds the static scratch" in str(ei.value)
    # tables that were never built: refused instead of built
    other = I.random_order(inst.n_vertices, 32)[:f]
    with pytest.raises(bb.BbtnError) as ei:
        h.region_bound_static(offs, verts, other, a1, out1)
    assert ei.value.status == bb.BBTN_EINVAL and "call bbtn_region_bound" in str(ei.value)
    h.close()
