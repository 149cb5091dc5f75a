"""bifrost_acc_static (include/bifrost.h): Eq. 6 with no context and no allocation - the scratch is a file-scope
static device array inside libbifrost.so.  Collected LAST (file name) so that, under `pytest -x`, nothing hides behind it.

Checked against the existing path (Context.acc) at the vector gate of the parity tests (normwise relative error
<= 1e-12), on calls in a row whose sizes change, so that what one call leaves in the shared array would show in the next."""
import numpy as np
import pytest

from conftest import normwise_rel_err, workload

TOL_VEC = 1e-12          # tests/test_gpu_parity.py's gate for acc


def _cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.mark.gpu
def test_acc_static_matches_the_context_path_on_calls_in_a_row():
    torch = _cuda()
    from paper_2210_02472_b200 import binding as B
    from paper_2210_02472_b200 import workloads as W
    torch.cuda.set_device(0)
    # 16384: the limit, packed path (pack -> pair -> finish);  5000: packed path, ragged;  3000 and 257: one fused launch
    sizes = [B.STATIC_MAX_N, 3000, 5000, 257, B.STATIC_MAX_N, 3000]
    cases = {}
    ctx = B.Context(B.STATIC_MAX_N)
    try:
        for n in sorted(set(sizes)):
            w = W.config4(n=n, n_sbh=max(1, n // 250), seed=100 + n)
            pos, mass = torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.mass).cuda()
            cases[n] = (w, pos, mass, ctx.acc(pos, mass, w.G, w.eps).cpu().numpy())
        torch.cuda.synchronize()
    finally:
        ctx.close()
    # outputs exist before the first call: the entry point and its binding allocate nothing
    outs = [torch.full((n, 3), float("nan"), dtype=torch.float64, device="cuda") for n in sizes]
    for n, out in zip(sizes, outs):       # back to back on one stream, no synchronisation in between
        w, pos, mass, _ = cases[n]
        assert B.acc_static(pos, mass, w.G, w.eps, out) is out
    torch.cuda.synchronize()
    for k, (n, out) in enumerate(zip(sizes, outs)):
        got, ref = out.cpu().numpy(), cases[n][3]
        assert np.isfinite(got).all(), f"call {k} (n = {n}) left rows unwritten"
        err = normwise_rel_err(got, ref)
        assert (err <= TOL_VEC).all(), f"call {k} (n = {n}): {err}"
    # the same input twice gives the same bits (fixed summation order, nothing read from the previous call)
    assert np.array_equal(outs[0].cpu().numpy(), outs[4].cpu().numpy())
    assert np.array_equal(outs[1].cpu().numpy(), outs[5].cpu().numpy())


@pytest.mark.gpu
def test_acc_static_against_the_oracle_and_its_limits():
    torch = _cuda()
    import oracle
    from paper_2210_02472_b200 import binding as B
    torch.cuda.set_device(0)
    w = workload(1)                                           # BASELINE configs[0]
    pos, mass = torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.mass).cuda()
    out = torch.empty((w.n, 3), dtype=torch.float64, device="cuda")
    for _ in range(2):
        out.fill_(float("nan"))
        B.acc_static(pos, mass, w.G, w.eps, out)
        err = normwise_rel_err(out.cpu().numpy(), oracle.acc(w.pos, w.mass, w.G, w.eps))
        assert (err <= TOL_VEC).all(), err
    # beyond the stated maximum: refused with a message that names the limit, nothing launched
    n = B.STATIC_MAX_N + 1
    big_pos = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
    big_mass = torch.ones(n, dtype=torch.float64, device="cuda")
    big_out = torch.full((n, 3), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(B.BifrostError, match="BIFROST_STATIC_MAX_N = 16384"):
        B.acc_static(big_pos, big_mass, 1.0, 0.0, big_out)
    torch.cuda.synchronize()
    assert bool((big_out == 7.0).all())
    # n = 0 is an empty call
    e = torch.empty((0, 3), dtype=torch.float64, device="cuda")
    B.acc_static(e, torch.empty(0, dtype=torch.float64, device="cuda"), 1.0, 0.0, e.clone())


@pytest.mark.gpu
def test_acc_static_takes_no_device_memory():
    """After one warm-up call per launch path, repeated calls leave the device's free memory where it was."""
    torch = _cuda()
    from paper_2210_02472_b200 import binding as B
    from paper_2210_02472_b200 import workloads as W
    torch.cuda.set_device(0)
    data = []
    for n in (B.STATIC_MAX_N, 2000):
        w = W.config4(n=n, n_sbh=8, seed=n)
        data.append((w, torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.mass).cuda(),
                     torch.empty((n, 3), dtype=torch.float64, device="cuda")))
    for w, pos, mass, out in data:
        B.acc_static(pos, mass, w.G, w.eps, out)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(0)
    for _ in range(20):
        for w, pos, mass, out in data:
            B.acc_static(pos, mass, w.G, w.eps, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(0)
    assert free1 >= free0, f"free device memory fell by {free0 - free1} bytes over 40 calls"


def test_static_entry_point_is_declared_and_exported():
    import os
    from paper_2210_02472_b200 import binding as B
    lib = B.load_library()
    assert hasattr(lib, "bifrost_acc_static") and hasattr(lib, "bifrost_static_error")
    header = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "bifrost.h")).read()
    assert f"#define BIFROST_STATIC_MAX_N {B.STATIC_MAX_N}" in header
    assert lib.bifrost_static_error() == b""
