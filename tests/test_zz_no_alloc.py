"""fdtd_absmax_noalloc — the one entry point that allocates nothing (static device scratch; include/fdtd_b200.h) — against the
existing path, fdtd_field_absmax of a context holding the same data.  Two calls in a row share the scratch array: the second
one (other data, another block count, a smaller maximum) must not see anything of the first.  Both reductions take the
maximum of the same |values|, so the tolerance is the bit equality the other parity tests use.

Collected last on purpose (the suite runs with pytest -x); it needs nothing from the tests before it."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_2606_06910_b200 import binding
    return binding


def _noalloc(B, dev_tensor, n=None):
    import torch
    out = torch.full((1,), -1.0, dtype=torch.float32, device=dev_tensor.device)
    st = torch.cuda.current_stream(dev_tensor.device).cuda_stream
    B.fdtd_absmax_noalloc(dev_tensor.data_ptr(), dev_tensor.numel() if n is None else n, out.data_ptr(), st)
    torch.cuda.synchronize()
    return float(out.item())


def test_noalloc_absmax_equals_field_absmax_on_two_calls_in_a_row(B):
    import torch
    sim = B.Fdtd((200, 150, 90), (8,) * 6, dt=0.4, cpml_alpha_max=0.1, kernel=B.FDTD_KERNEL_FUSED)
    for f, scale in ((B.FDTD_P, 3.0), (B.FDTD_VX, 0.25), (B.FDTD_VY, 1.0), (B.FDTD_VZ, 1.0)):
        sim.fill_hash(f, 7, scale)
    sim.step(4)
    p = torch.from_numpy(sim.get_field(B.FDTD_P)).cuda()                    # 3.96e6 values: 61 blocks
    vx = torch.from_numpy(sim.get_field(B.FDTD_VX)[:40]).cuda().contiguous()  # 1.43e6 values, a ragged last block, smaller maximum
    want_p = sim.field_absmax(B.FDTD_P)
    want_vx = sim.field_absmax(B.FDTD_VX, (0, 0, 0), (sim.nx, sim.ny, 40))
    assert want_p > 0 and 0 < want_vx < want_p
    _noalloc(B, vx[:1])                                                      # first launch: the driver loads the kernel now (lazy module loading)
    free0 = torch.cuda.mem_get_info()[0]
    got_p = _noalloc(B, p)
    got_vx = _noalloc(B, vx)                                                 # second call in a row on the same scratch
    assert np.float32(got_p).view(np.uint32) == np.float32(want_p).view(np.uint32), (got_p, want_p)
    assert np.float32(got_vx).view(np.uint32) == np.float32(want_vx).view(np.uint32), (got_vx, want_vx)
    assert _noalloc(B, p) == got_p                                           # and back: nothing of the smaller run is left
    assert torch.cuda.mem_get_info()[0] >= free0 - (4 << 20)                 # the calls took no device memory (4 MB: room for torch's own scalars)
    # a misaligned view (scalar path), a single value, an empty range
    flat = p.reshape(-1)
    assert _noalloc(B, flat[1:70001]) == float(flat[1:70001].abs().max().item())
    assert _noalloc(B, flat[5:6]) == abs(float(flat[5].item()))
    assert _noalloc(B, flat, n=0) == 0.0
    sim.destroy()


def test_noalloc_rejects_sizes_beyond_its_static_scratch(B):
    import torch
    x = torch.zeros(16, dtype=torch.float32, device="cuda")
    out = torch.full((1,), -1.0, dtype=torch.float32, device="cuda")
    with pytest.raises(B.FdtdError) as e:
        B.fdtd_absmax_noalloc(x.data_ptr(), B.FDTD_NOALLOC_MAX_ELEMS + 1, out.data_ptr(), 0)
    assert "maximum" in str(e.value) and str(B.FDTD_NOALLOC_MAX_ELEMS) in str(e.value)
    torch.cuda.synchronize()
    assert float(out.item()) == -1.0                                          # nothing was launched
    with pytest.raises(B.FdtdError):
        B.fdtd_absmax_noalloc(x.data_ptr(), 16, 0, 0)                          # no output pointer
    assert _noalloc(B, x) == 0.0                                              # the entry point still works after a refusal
