"""chime_bf_dedisperse_beams_noalloc: the dedispersion kernel with its scratch (the delay table) in the library's
built-in device array, for callers that cannot allocate device memory.  Expected values: the existing path,
chime_bf_dedisperse_beams with a caller-owned table (itself bit-exact against the oracle in tests/test_gpu_dedisp.py).
Integer work: the comparison is bit-exact.  This file is collected last on purpose (the suite runs with pytest -x)."""
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


def _case(bf, seed, C, R, nb, dm, upchan_len):
    g = torch.Generator(device="cuda").manual_seed(seed)
    beams = torch.randint(0, 256, (C, R, nb, 16), dtype=torch.uint8, device="cuda", generator=g)
    freqs = 800.0 - 0.390625 * (np.arange(C) * (1024 // C))        # spread over the band: distinct delays per channel
    want = bf.dedisperse_beams(beams, freqs, dm, upchan_len=upchan_len)   # existing path (allocates its table)
    torch.cuda.synchronize()
    out = torch.full(tuple(want.shape), -12345, dtype=torch.int32, device="cuda")   # garbage: the call must not rely on zeros
    bf.dedisperse_beams_noalloc(beams, freqs, dm, out, upchan_len=upchan_len)
    torch.cuda.synchronize()
    assert torch.equal(out, want), (C, R, nb, dm, int((out != want).sum()))
    return int(want.shape[1])


def test_noalloc_matches_existing_path_two_calls_in_a_row(bf):
    """Two calls in a row share the built-in array: the second one (fewer channels, another DM, another frame length)
    finds the first one's table in it and must not be disturbed by it.  The first case is small enough in beams x time
    for the channel loop to be split over blockIdx.z (atomicAdd into a cleared output)."""
    n1 = _case(bf, 1, C=12, R=96, nb=32, dm=3.0, upchan_len=128)
    n2 = _case(bf, 2, C=5, R=64, nb=64, dm=4.0, upchan_len=256)
    assert n1 >= 1 and n2 >= 1
    # and once more with the first shape: the table is rewritten, not accumulated
    _case(bf, 3, C=12, R=96, nb=32, dm=3.0, upchan_len=128)


def test_noalloc_allocates_nothing_on_the_device(bf):
    C, R, nb = 4, 48, 32
    beams = torch.randint(0, 256, (C, R, nb, 16), dtype=torch.uint8, device="cuda")
    freqs = 800.0 - 0.390625 * np.arange(C)
    out = torch.empty((nb, R), dtype=torch.int32, device="cuda")
    bf.dedisperse_beams_noalloc(beams, freqs, 0.0, out)      # first call on this device: the address lookup happens here
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        bf.dedisperse_beams_noalloc(beams, freqs, 0.0, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    assert torch.equal(out, beams.to(torch.int32).sum(dim=(0, 3)).transpose(0, 1).contiguous())   # DM 0: plain sums


def test_noalloc_rejects_sizes_beyond_the_built_in_scratch(bf):
    C = bf.NOALLOC_MAX_COARSE + 1
    beams = torch.zeros((C, 2, 32, 16), dtype=torch.uint8, device="cuda")
    out = torch.empty((32, 2), dtype=torch.int32, device="cuda")
    with pytest.raises(bf.ChimeBfError, match="exceeds the built-in scratch"):
        bf.dedisperse_beams_noalloc(beams, np.full(C, 600.0), 0.0, out)
