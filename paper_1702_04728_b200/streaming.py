"""Full-band streaming (BASELINE.json configs[3]): the 1024 coarse
channels of one 49152-sample chunk are processed as channel groups (default 8 x 128 channels, 12.9 GB of
packed baseband each) through two device buffers on two CUDA streams (ping-pong): while group g executes
on one stream, the other stream's buffer is being refilled for group g+1.  Channels are independent
(PAPER.md:47, :53), so the groups need no exchange; each group has its own plan (its own frequencies,
index tables and folded weights).

Stream and buffer plumbing only: every step of the beamformer runs inside chime_bf_execute.
"""
import numpy as np

from . import N_INPUT, plan_create_ex


class FullBandStreamer:
    def __init__(self, n_coarse=1024, group=128, n_time=49152, freq_mhz=None, gains=None, zero_pad=512,
                 upchan_len=128, n_buffers=2, alloc_input=True):
        import torch
        if n_coarse % group:
            raise ValueError("n_coarse must be a multiple of the channel group size")
        if freq_mhz is None:
            freq_mhz = 800.0 - 0.390625 * np.arange(n_coarse)
        freq_mhz = np.asarray(freq_mhz, dtype=np.float64)
        self.n_coarse, self.group, self.n_time = n_coarse, group, n_time
        self.n_groups = n_coarse // group
        self.plans = []
        for g in range(self.n_groups):
            sl = slice(g * group, (g + 1) * group)
            self.plans.append(plan_create_ex(group, freq_mhz=freq_mhz[sl],
                                             gains=None if gains is None else gains[sl],
                                             zero_pad=zero_pad, upchan_len=upchan_len, n_time=n_time))
        self.streams = [torch.cuda.Stream() for _ in range(n_buffers)]
        self.in_bufs = ([torch.empty((group, n_time, N_INPUT), dtype=torch.uint8, device="cuda")
                         for _ in range(n_buffers)] if alloc_input else None)
        self.group_in_bytes = group * n_time * N_INPUT
        self.group_out_shape = self.plans[0].out_shape
        self.launches = 0

    def run_chunk(self, fill, out_u8=None, out_f32=None):
        """One full-band chunk.  fill(g, buf) writes group g's packed baseband [group][n_time][2048] into
        `buf` (it is called with that buffer's stream current; None = reuse what the buffers hold).
        out_u8 / out_f32: optional lists of per-group output tensors (allocated when None and returned).
        Asynchronous: call synchronize() before reading the outputs."""
        import torch
        nb = len(self.streams)
        if out_u8 is None:
            out_u8 = [torch.empty(self.group_out_shape, dtype=torch.uint8, device="cuda")
                      for _ in range(self.n_groups)]
        for g, plan in enumerate(self.plans):
            s, buf = self.streams[g % nb], self.in_bufs[g % nb]
            with torch.cuda.stream(s):
                if fill is not None:
                    fill(g, buf)
                plan.execute(buf, out_u8[g], stream=s)
                self.launches += plan.launches_per_execute
                if out_f32 is not None:
                    plan.execute_f32(buf, out_f32[g], stream=s)
                    self.launches += plan.launches_per_execute
        return out_u8

    def synchronize(self):
        for s in self.streams:
            s.synchronize()

    def destroy(self):
        for p in self.plans:
            p.destroy()
        self.plans = []
