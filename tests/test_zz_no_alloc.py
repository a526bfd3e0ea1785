"""mc_energy_noalloc: the entry point for callers that cannot allocate device memory (include/mcb200.h).  Its
output is compared with the existing path's (mc_init + mc_energy) on two calls in a row, which share the static
scratch array.  Collected last on purpose (the suite runs with pytest -x).  Inputs are seeded and synthetic."""
import re
from pathlib import Path

import numpy as np
import pytest

from paper_1602_05716_b200 import workloads as W

ROOT = Path(__file__).resolve().parents[1]
E_RTOL = 1e-9     # the energy tolerance of the parity tests


def test_noalloc_entry_point_calls_no_allocator():
    """Host logic: the body of mc_energy_noalloc contains no allocating call, takes the scratch address from
    cudaGetSymbolAddress and checks its return code; the scratch array is a static __device__ array."""
    src = (ROOT / "paper_1602_05716_b200" / "csrc" / "mcb200.cu").read_text()
    body = src[src.index('extern "C" int mc_energy_noalloc('):]
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMemPool", "cudaStreamCreate", "cudaEventCreate", "new ",
                   "std::vector", "malloc("):
        assert banned not in body, banned
    assert "cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch)" in body and "e != cudaSuccess" in body
    assert re.search(r"static __device__ __align__\(256\) double g_noalloc_scratch\[kNoAllocMaxUnits\];", src)
    hdr = (ROOT / "include" / "mcb200.h").read_text()
    assert "#define MC_NOALLOC_MAX_N 131072" in hdr


@pytest.mark.gpu
def test_noalloc_energy_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    torch.cuda.set_device(0)
    from paper_1602_05716_b200.binding import MCError, MCSystem, load_library, mc_energy_noalloc
    load_library()
    dev = torch.device("cuda", 0)
    out = torch.zeros(1, dtype=torch.float64, device=dev)

    # two systems of different size (the second call finds the first call's partials in the scratch array): a ragged
    # N that spans several 1024-row blocks with a partly filled last tile, then a small one inside one block
    cases = [W.scaled(W.CONFIGS[2], 5000), W.scaled(W.CONFIGS[0], 700)]
    refs, inputs = [], []
    for w in cases:
        pos, q, d = w.arrays()
        g = MCSystem(pos, q, d, w.cavity_R, w.bjerrum, w.max_disp, w.seed, validate=False)
        g.mc_set_positions(pos)
        g.mc_sweep(2)                                   # a configuration the chain produced, not only the initial one
        refs.append(g.mc_energy())
        inputs.append((g.mc_get_positions().clone(), torch.from_numpy(np.ascontiguousarray(q, dtype=np.float64)).to(dev),
                       w.bjerrum))
        g.close()
    torch.cuda.synchronize()
    got = []
    free_before = None
    for k, (p, qd, lb) in enumerate(inputs + inputs):    # four calls back to back on one stream
        if k == 2:
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]   # kernels are loaded by now: later calls must not take memory
        mc_energy_noalloc(p, qd, lb, out)
        got.append(out.clone())
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "a call allocated device memory"
    got = [float(x.item()) for x in got]
    for k, e in enumerate(got):
        ref = refs[k % 2]
        assert np.isfinite(e) and abs(e - ref) <= E_RTOL * max(abs(ref), 1.0), (k, e, ref)
    assert got[0] == got[2] and got[1] == got[3], "the result depends on what the scratch array held before"

    # beyond the stated maximum: refused with a clear error, nothing launched
    n_big = 131072 + 1
    with pytest.raises(MCError) as ei:
        load_library()   # (keeps the library handle warm; the call below is the one that must fail)
        big_p = torch.zeros((3, n_big), dtype=torch.float64, device=dev)
        big_q = torch.zeros(n_big, dtype=torch.float64, device=dev)
        mc_energy_noalloc(big_p, big_q, 1.0, out)
    assert ei.value.code == -4 and "MC_NOALLOC_MAX_N" in str(ei.value)
    torch.cuda.synchronize()
