"""Error behaviour of the C-ABI on a GPU box (include/chime_bf.h: "Returns NULL on error", negative codes)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bf():
    import __graft_entry__ as g
    g.build()
    import paper_1702_04728_b200 as bf
    return bf


@pytest.mark.parametrize("kw,msg", [
    (dict(zero_pad=384), "zero_pad"), (dict(upchan_len=64), "upchan_len"), (dict(n_time=1000), "n_time"),
    (dict(n_time=0), "n_time"), (dict(n_coarse=0), "n_coarse"), (dict(upchan_len=256, n_time=384), "n_time"),
])
def test_plan_creation_rejects_bad_parameters(bf, kw, msg):
    args = dict(n_coarse=1, n_time=384)
    args.update(kw)
    n = args.pop("n_coarse")
    with pytest.raises(bf.ChimeBfError, match=msg):
        bf.plan_create_ex(n, **args)


def test_execute_rejects_misaligned_and_null_buffers(bf):
    plan = bf.plan_create_ex(1, n_time=384)
    lib = bf.load_library()
    buf = torch.zeros(plan.in_bytes + 16, dtype=torch.uint8, device="cuda")
    out = torch.zeros(plan.out_elems + 16, dtype=torch.uint8, device="cuda")
    assert lib.chime_bf_execute(plan._h, None, buf.data_ptr() + 1, out.data_ptr()) == -2      # E_ALIGNMENT
    assert "aligned" in bf.last_error()
    assert lib.chime_bf_execute(plan._h, None, buf.data_ptr(), out.data_ptr() + 4) == -2
    assert lib.chime_bf_execute(plan._h, None, None, out.data_ptr()) == -1                     # E_INVALID_ARG
    assert lib.chime_bf_execute(None, None, buf.data_ptr(), out.data_ptr()) == -1
    assert lib.chime_bf_execute(plan._h, None, buf.data_ptr(), out.data_ptr()) == 0
    torch.cuda.synchronize()
    with pytest.raises(ValueError):
        plan.execute(torch.zeros(100, dtype=torch.uint8, device="cuda"))                       # wrong size (binding)
    lib.chime_bf_destroy(None)                                                                 # NULL-safe
    plan.destroy()
    plan.destroy()                                                                             # idempotent


def test_nibble_zero_decodes_to_minus_eight(bf, orc):
    """Reading A1: nibble 0 is arithmetic -8, not a flag -- the generators never emit it, the kernels must still
    agree with the oracle on it (all-zero bytes = every sample at -8-8i)."""
    plan = bf.plan_create_ex(1, freq_mhz=[700.0], n_time=384)
    z = torch.zeros((1, 384, 2048), dtype=torch.uint8, device="cuda")
    z[0, ::7, ::3] = 0x0F
    got = plan.execute_f32(z).cpu().numpy()[0, 0]
    I, _ = orc.cell(z[0].cpu().numpy(), 700.0)
    mean = I.mean(axis=-1, keepdims=True)                      # north star: 1e-4 of each beam's mean power
    assert (np.abs(got - I) / mean).max() <= 1e-4
    q = plan.execute(z).cpu().numpy()[0, 0]
    assert np.abs(q.astype(int) - orc.quantize(I).astype(int)).max() <= 1 and q.max() == 255
    plan.destroy()
