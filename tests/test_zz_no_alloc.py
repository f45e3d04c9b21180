"""prs_diagnostics_static: the wall diagnostics for callers that must not allocate (include/prs.h, csrc/prs_static.cu).

The entry point takes caller-held device fields and a 24-byte device record, uses a static __device__ scratch array
inside the library (786 688 bytes, at most 2^27 sites) and calls no allocating routine.  Checked here against the
existing path (prs_diagnostics on a handle, itself checked against the oracle in test_gpu_parity.py): counts equal,
the velocity sum within the 1e-10 relative bar the other diagnostics tests use, on calls in a row that share the array.

This file sorts last on purpose (pytest -x: a failure here hides nothing after it) and passes both
alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

import paper_1710_10420_b200 as prs
from paper_1710_10420_b200 import prs as binding


def test_static_scratch_limits_and_rejection_need_no_gpu():
    """The stated size and limit, and the refusal of larger lattices, which happens before any CUDA call."""
    L = prs.lib()
    assert L.prs_diagnostics_static_scratch_bytes() == 256 + 24 * 32768 == 786688
    assert L.prs_diagnostics_static_max_sites() == 1 << 27
    for dims, N in ((2, 11586), (3, 513), (3, 8192), (2, 1 << 20)):
        assert N ** dims > 1 << 27
        with pytest.raises(prs.PrsError) as e:
            binding.diagnostics_static(dims, N, prs.F32, 256, 256, 256)          # never dereferenced
        assert e.value.code == 2 and "maximum of 134217728" in str(e.value)
    for bad in ((4, 8, prs.F32), (2, 0, prs.F32), (2, 8, 7)):
        with pytest.raises(prs.PrsError) as e:
            binding.diagnostics_static(bad[0], bad[1], bad[2], 256, 256, 256)
        assert e.value.code == 1
    with pytest.raises(prs.PrsError) as e:
        binding.diagnostics_static(2, 8, prs.F32, None, 256, 256)
    assert e.value.code == 1


def read_sums(out):
    host = out.cpu().numpy()
    return int(host[0]), int(host[1]), float(host[2:3].view(np.float64)[0])


@pytest.mark.gpu
@pytest.mark.parametrize("dims,N,prec", [(2, 1000, prs.F32), (2, 4097, prs.F64), (3, 128, prs.F32), (3, 101, prs.F64),
                                         (2, 3, prs.F32), (3, 512, prs.F32)])
def test_static_diagnostics_match_the_handle_path_on_calls_in_a_row(dims, N, prec):
    import torch

    g = prs.Simulation(dims, N, prec, seed=5)
    g.init(1.0)
    out = torch.empty(3, dtype=torch.int64, device="cuda")
    stream = torch.cuda.current_stream()
    seen = []
    # several calls in a row on different states (white noise, forming, formed network): the shared static array keeps
    # the previous call's partials and must not leak them into the next result
    for nsteps in (0, 30, 200 if N <= 1000 else 40):
        g.step(nsteps)
        want = g.diagnostics()
        p, v = g.device_pointers()
        out.fill_(-1)                                            # stale output must be overwritten
        binding.diagnostics_static(dims, N, prec, p, v, out, stream)
        links, walls, ratio = read_sums(out)
        assert links == want["link_count"] and walls == want["wall_sites"], (nsteps, links, walls, want)
        assert abs(ratio - want["sum_ratio"]) <= 1e-10 * max(want["sum_ratio"], 1e-300)
        # the same state again, back to back: same launch configuration, same summation order -> the same bits
        out.fill_(-1)
        binding.diagnostics_static(dims, N, prec, p, v, out, stream)
        assert read_sums(out) == (links, walls, ratio)
        # rho and gv2 from the three sums through the library's own normalisation
        d = binding.diag_combine([{"step": want["step"], "eta": want["eta"], "link_count": links, "wall_sites": walls,
                                   "sum_ratio": ratio}], dims, N)
        assert d["rho"] == want["rho"] and abs(d["gv2"] - want["gv2"]) <= 1e-10 * max(want["gv2"], 1e-300)
        seen.append(links)
    assert len(set(seen)) == len(seen)                           # the states really differed
    g.close()


@pytest.mark.gpu
def test_static_diagnostics_on_caller_tensors_and_a_stream_of_its_own():
    """Fields that never belonged to a handle (plain torch tensors), a non-default stream, and a large lattice right
    before a small one (the small pass must not see the large one's partials)."""
    import torch
    from oracle import binding as ref
    from tests import fieldgen as fg

    st = torch.cuda.Stream()
    out = torch.empty(3, dtype=torch.int64, device="cuda")
    for dims, N in ((2, 2048), (2, 64), (3, 160), (3, 8)):
        phi, pd = fg.random_state(dims, N, 21, np.float32, amp=1.5)
        tp, tv = torch.from_numpy(phi).cuda(), torch.from_numpy(pd).cuda()
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            binding.diagnostics_static(dims, N, prs.F32, tp, tv, out, st)
        st.synchronize()
        links, walls, ratio = read_sums(out)
        want = ref.diagnostics_of(phi, pd)                       # the oracle on the same bytes
        assert links == want["link_count"] and walls == want["wall_sites"]
        assert abs(ratio - want["sum_ratio"]) <= 1e-10 * want["sum_ratio"]
    with pytest.raises(prs.PrsError) as e:
        binding.diagnostics_static(2, 64, prs.F32, phi, tv, out, st)            # a host array is not a device pointer
    assert e.value.code == 1
