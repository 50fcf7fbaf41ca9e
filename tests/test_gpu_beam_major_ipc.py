"""The peer-pointer path of chime_bf_execute_beam_major with a REAL second process: rank 1 runs in a child process
and stores its beams through CUDA-IPC mappings of receive buffers that live in the parent's address space (what a
peer-mapped NVLink buffer is to the kernel: a device pointer that belongs to somebody else).  One GPU is enough; the two
processes' kernels never wait on one another.  Expected values: the oracle."""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu

W, C_LOCAL, R, U = 2, 1, 2, 128


def _rank_work(rank, recv, ready, done, err):
    try:
        import __graft_entry__ as g
        g.build()
        import paper_1702_04728_b200 as bf
        T = R * 3 * U
        seed = synth.config_seed(3) + 99
        freqs = synth.chime_freqs_mhz(W * C_LOCAL, 211)
        gains = synth.gains(seed, W * C_LOCAL, flagged_frac=0.03)
        d_in = synth.noise_bytes(seed, W * C_LOCAL, T, device="cuda")
        sl = slice(rank * C_LOCAL, (rank + 1) * C_LOCAL)
        plan = bf.plan_create_ex(C_LOCAL, freq_mhz=freqs[sl], gains=gains[sl], n_time=T)
        plan.execute_beam_major(d_in[sl].contiguous(), recv, chan_global0=rank * C_LOCAL)
        torch.cuda.synchronize()
        assert plan.kernel_status() == 0
        plan.destroy()
        done.put(rank)
    except Exception as e:      # pragma: no cover
        err.put(repr(e))
        done.put(-1)


def test_beam_major_through_ipc_mapped_buffers(orc):
    import torch.multiprocessing as mp
    from paper_1702_04728_b200 import beam_major
    ctx = mp.get_context("spawn")
    C_total, T = W * C_LOCAL, R * 3 * U
    recv = [torch.full(beam_major.receive_shape(C_total, R, W), 0xEE, dtype=torch.uint8, device="cuda") for _ in range(W)]
    torch.cuda.synchronize()
    ready, done, err = ctx.Queue(), ctx.Queue(), ctx.Queue()
    child = ctx.Process(target=_rank_work, args=(1, recv, ready, done, err))   # CUDA tensors travel as IPC handles
    child.start()
    _rank_work(0, recv, ready, done, err)                                       # rank 0 in this process, local pointers
    got = sorted(done.get(timeout=300) for _ in range(2))
    child.join(timeout=60)
    assert got == [0, 1], err.get() if not err.empty() else got
    torch.cuda.synchronize()
    host = [x.cpu().numpy() for x in recv]
    seed = synth.config_seed(3) + 99
    freqs = synth.chime_freqs_mhz(C_total, 211)
    gains = synth.gains(seed, C_total, flagged_frac=0.03)
    hb = synth.noise_bytes(seed, C_total, T).numpy()
    n_diff = n_tot = 0
    for cg in range(C_total):
        for Rf in range(R):
            I, _ = orc.cell(hb[cg, 384 * Rf:384 * (Rf + 1)], float(freqs[cg]), gains=gains[cg])
            q = orc.quantize(I).reshape(1024, 16)
            for d in range(W):
                b0, nb = beam_major.beam_shard(W, d)
                diff = np.abs(host[d][cg, Rf].astype(int) - q[b0:b0 + nb].astype(int))
                assert diff.max() <= 1
                n_diff += int((diff != 0).sum())
                n_tot += diff.size
    assert n_diff <= 1e-3 * n_tot


def test_peer_buffer_ptrs_single_rank():
    from paper_1702_04728_b200 import beam_major
    buf = torch.zeros(beam_major.receive_shape(1, 1, 1), dtype=torch.uint8, device="cuda")
    assert beam_major.peer_buffer_ptrs(buf) == [buf.data_ptr()]
