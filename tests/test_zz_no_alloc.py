"""gcoreccd_field_noalloc (include/gcoreccd.h): eq. 6 with no handle and no device allocation — its scratch is a
file-scope `static __device__` array inside the library — against the existing path (load_carriers + eval_field on a
handle), on calls in a row that share that array.  Collected last (the file name), so that a failure here hides no other
test from `pytest -x`."""
import numpy as np
import pytest

import workloads
from util import field_rel_err, gpu_sim

FIELD_TOL = 1e-4          # north_star: per-carrier field vectors within 1e-4 relative (tests/test_gpu_parity.py)


def test_sizes_beyond_the_fixed_scratch_are_refused_without_touching_a_gpu():
    from paper_2203_11043_b200 import binding as b
    with pytest.raises(b.GcoreccdError) as e:
        b.field_noalloc(0, b.NOALLOC_MAX_CARRIERS + 1, 1e-3, 11.7, 0)
    assert e.value.code == b.ERR_CAPACITY and "GCORECCD_NOALLOC_MAX_CARRIERS = 16384" in str(e.value)
    b.field_noalloc(0, 0, 1e-3, 11.7, 0)                                       # n = 0: a no-op, even with null pointers
    with pytest.raises(b.GcoreccdError) as e:
        b.field_noalloc(0, 5, 1e-3, 11.7, 0)
    assert e.value.code == b.ERR_INVALID


def _existing_path(w):
    """Field of the holes a handle holds after the load (a track's hole at the collection plane is collected at once and
    feels no field), in the handle's order: (xyz, E)."""
    sim = gpu_sim(w)
    sim.load_carriers(w["xyz"])
    xyz, _ = sim.read_carriers()
    E = sim.eval_field()
    sim.close()
    return np.ascontiguousarray(xyz, dtype=np.float32), E


@pytest.mark.gpu
def test_allocation_free_field_equals_the_existing_path_on_calls_in_a_row():
    import torch
    from paper_2203_11043_b200 import binding as b
    stream = torch.cuda.Stream()
    # a large call first, then smaller ones: whatever the first leaves in the shared array (positions beyond n, partial
    # sums of more chunks, its plan) must not reach a later result; sizes hit all three field variants and a ragged tail
    cases = [(1, 16384), (3, 5000), (0, 777), (2, 12289), (0, 1)]
    ws = [workloads.make(cfg, n=n) for cfg, n in cases]
    refs = [(w,) + _existing_path(w) for w in ws]                              # (workload, xyz of the active holes, E)
    xin = [torch.from_numpy(x).cuda() for _, x, _ in refs]
    out = [torch.full((len(x), 3), float("nan"), dtype=torch.float32, device="cuda") for _, x, _ in refs]
    torch.cuda.synchronize()

    def run(k):
        P = refs[k][0]["params"]
        b.field_noalloc(xin[k].data_ptr(), len(refs[k][1]), P["softening_um"], P["eps_si"], out[k].data_ptr(), stream.cuda_stream)

    run(0)                                                                     # (first call on the device: set-up)
    stream.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for k in range(1, len(cases)):                                             # back to back on one stream, no sync between
        run(k)
    run(0)
    stream.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                               # nothing was allocated by those calls
    first = out[0].cpu().numpy().copy()
    for k, (w, _, E_ref) in enumerate(refs):
        E = out[k].cpu().numpy()
        assert np.isfinite(E).all()
        if len(E) > 1:
            rel, _ = field_rel_err(E, E_ref.astype(np.float64))
            assert rel <= FIELD_TOL, (cases[k], rel)
        else:
            assert np.array_equal(E, np.zeros((1, 3), dtype=np.float32))       # a lone hole feels no field (self term 0)
    # the same input again gives the same bits (fixed plan, fixed summation order), whatever ran in between
    out[0].fill_(float("nan"))
    run(0)
    stream.synchronize()
    assert np.array_equal(out[0].cpu().numpy(), first)
