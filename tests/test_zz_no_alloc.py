"""tpcclus_pack_noalloc (include/tpcclus.h): the packed output of an ordered cluster list without a handle, a
workspace or any allocation -- its scratch is a static array in device memory that all calls share and that keeps
the last call's contents.  Checked byte for byte against the existing path (tpcclus_run_packed) on two calls in a
row with different frames, so that anything the first call leaves in the array would show in the second.

Collected last on purpose (the file name): the suite runs with pytest -x."""
import numpy as np
import pytest

from workloads import make_frame

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tp(cuda_device):
    import paper_2511_17018_b200 as tp
    tp.lib()   # fails loudly if the extension is missing
    return tp


def _reference(tp, fr, dev):
    """(32-byte deterministic clusters, packed clusters, row index, n) of frame `fr` from the existing path."""
    import torch
    c = tp.Clusterizer(fr.n_sectors, fr.n_rows, fr.n_time, fr.n_pads, fr.n_digits)
    d = fr.digits.to(dev)
    packed, ridx, nt, st = c.run_packed(d)
    torch.cuda.synchronize()
    n = int(nt.item())
    assert int(st.item()) == 0 and n > 100
    packed, ridx = packed[:n].clone(), ridx.clone()
    cl, nt, st = c.run(d, tp.MODE_DETERMINISTIC)
    torch.cuda.synchronize()
    assert int(nt.item()) == n
    cl = cl[:n].clone()
    c.close()
    return cl, packed, ridx, n


def test_pack_noalloc_matches_run_packed_on_two_calls_in_a_row(tp, cuda_device):
    import torch
    frames = [make_frame(0), make_frame(4, device=cuda_device, sectors=[0, 7, 35], n_time=300), make_frame(1)]
    refs = [(fr, *_reference(tp, fr, cuda_device)) for fr in frames]
    # every buffer exists before the first call: the calls below allocate nothing, on the device or through torch
    outs = [(torch.full((n, 16), 0xAB, dtype=torch.uint8, device=cuda_device),
             torch.full((fr.n_sectors * fr.n_rows + 1,), -1, dtype=torch.int64, device=cuda_device)) for fr, _, _, _, n in refs]
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream(cuda_device).cuda_stream
    before = torch.cuda.memory_allocated(cuda_device)
    for rep in range(2):       # the whole sequence twice: frames of 152, 456 and 16 (sector,row) pairs after one another
        for (fr, cl, _, _, n), (o_packed, o_ridx) in zip(refs, outs):
            tp.tpcclus_pack_noalloc(cl.data_ptr(), n, fr.n_sectors, fr.n_rows, o_packed.data_ptr(), o_ridx.data_ptr(), stream)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated(cuda_device) == before
        for (fr, cl, packed, ridx, n), (o_packed, o_ridx) in zip(refs, outs):
            assert o_packed.cpu().numpy().tobytes() == packed.cpu().numpy().tobytes(), (rep, fr.n_rows)
            assert torch.equal(o_ridx, ridx), (rep, fr.n_rows)
            o_packed.fill_(0xCD)
            o_ridx.fill_(-7)
        torch.cuda.synchronize()
    # an empty list: the index is all zero
    fr, cl, _, _, n = refs[0]
    o_packed, o_ridx = outs[0]
    tp.tpcclus_pack_noalloc(0, 0, fr.n_sectors, fr.n_rows, 0, o_ridx.data_ptr(), stream)
    torch.cuda.synchronize()
    assert int(o_ridx.abs().sum().item()) == 0


def test_pack_noalloc_refuses_what_the_static_scratch_cannot_hold(tp, cuda_device):
    import torch
    ridx = torch.zeros(8, dtype=torch.int64, device=cuda_device)
    buf = torch.zeros((4, 32), dtype=torch.uint8, device=cuda_device)
    out = torch.zeros((4, 16), dtype=torch.uint8, device=cuda_device)
    for S, R, n, word in ((257, 256, 4, "scratch"), (300, 300, 4, "scratch"), (0, 4, 4, "scratch"), (1, 4, 1 << 32, "maximum")):
        with pytest.raises(tp.TpcclusError) as e:
            tp.tpcclus_pack_noalloc(buf.data_ptr(), n, S, R, out.data_ptr(), ridx.data_ptr(), 0)
        assert e.value.code == -1 and word in str(e.value) and "tpcclus_pack_noalloc" in str(e.value)
    with pytest.raises(tp.TpcclusError) as e:   # misaligned output
        tp.tpcclus_pack_noalloc(buf.data_ptr(), 4, 1, 4, out.data_ptr() + 4, ridx.data_ptr(), 0)
    assert e.value.code == -1 and "misaligned" in str(e.value)
    torch.cuda.synchronize()
