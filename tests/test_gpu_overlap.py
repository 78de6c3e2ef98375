"""GPU parity of the S7 stream-overlap harness (SURVEY 8(a) S7; PAPER.md:61, :477 "Wait time", :505 "We reserved only 64 SMs
for decompression"): batch i+1's fetch+decode on one stream against a consumer of batch i on another, two buffers.

What can go wrong silently in a double-buffered schedule is a STALE or HALF-OVERWRITTEN buffer: the consumer of step i reading
buffer i % 2 before fetch(i) finished, or fetch(i+2) overwriting it before consume(i) finished.  So the consumer here COPIES the
buffer into a per-step result tensor, every step fetches different rows, and every step's bytes are compared with the plain
gather of the original rows (oracle (c1)) and, on a sample, with the oracle codec (c2).  Both orderings are exercised: a fast
consumer (the fetch is the long leg: the consumer waits on fetched[i]) and a slow consumer (a spin kernel in front of the copy:
the fetch runs ahead and must wait on consumed[i-2]).  The decode grid is limited with ibp_configure(max_ctas) to 8, 32 and the
library default, the SM share being a launch parameter of the persistent kernels.
"""
import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import workloads
from paper_2605_30728_b200.overlap import DoubleBufferedPipeline

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

N_STEPS = 7


def _u8(X):
    X = np.ascontiguousarray(X)
    return X.view(np.uint8).reshape(X.shape[0], -1)


def _run(pipe_fetch, buf_rows, row_bytes, n_steps, slow_consumer):
    bufs = [torch.full((buf_rows, row_bytes), 0xEE, dtype=torch.uint8, device="cuda") for _ in range(2)]
    results = [torch.full((buf_rows, row_bytes), 0x11, dtype=torch.uint8, device="cuda") for _ in range(n_steps)]

    def fetch(i, bi, stream_ptr):
        pipe_fetch(i, bufs[bi], stream_ptr)

    def consume(i, bi):
        if slow_consumer:
            torch.cuda._sleep(3_000_000)                       # ~1.5 ms spin: the fetch of steps i+1, i+2 catches up and must wait
        results[i].copy_(bufs[bi])
        bufs[bi].fill_(0xEE)                                   # poison after use: a fetch that did not really rewrite the buffer shows

    pipe = DoubleBufferedPipeline(fetch, consume, n_steps)
    ms = pipe.run_overlapped()
    torch.cuda.synchronize()
    assert ms > 0
    return [r.cpu().numpy() for r in results]


@pytest.mark.parametrize("max_ctas", [8, 32, 0])
@pytest.mark.parametrize("slow_consumer", [False, True])
def test_overlapped_weight_layers(max_ctas, slow_consumer):
    """configs[4] in small: three distinct 'layers' of two bf16 matrices each (strided groups = 128-column tiles), streamed in
    order with ibp_gather_decompress_range, one layer per step, 7 steps."""
    shapes = [(384, 512), (256, 1408)]
    layers = []
    for l in range(3):
        mats = []
        for s, (r, c) in enumerate(shapes):
            wm = workloads.WeightMatrix(r, c, layer=l, slot=s)
            X = wm.table()
            h = ibp.ibp_build(X, 256, 1, wm.group_param, align_bytes=16).upload_metadata(0)
            if max_ctas:
                h.configure(max_ctas, 0)
            mats.append((h, wm.n_rows, _u8(X)))
        layers.append(mats)
    layer_rows = sum(m[1] for m in layers[0])

    def fetch(i, buf, stream_ptr):
        off = 0
        for h, n_rows, _ in layers[i % 3]:
            h.gather_decompress_range(0, n_rows, buf.data_ptr() + off * 256, stream_ptr)
            off += n_rows

    got = _run(fetch, layer_rows, 256, N_STEPS, slow_consumer)
    for i in range(N_STEPS):
        want = np.concatenate([m[2] for m in layers[i % 3]])
        assert np.array_equal(got[i], want), f"step {i}: the consumer saw a stale or half-written buffer"
    # (c2): the oracle codec on the first matrix of layer 1
    h, n_rows, Xb = layers[1][0]
    ds = oracle.Dataset(Xb, 1, shapes[0][1] // 128)
    ids = np.arange(0, n_rows, 37, dtype=np.int64)
    assert np.array_equal(got[1][ids], ds.gather_decompress(ids))
    ds.close()
    for mats in layers:
        for m in mats:
            m[0].destroy()


@pytest.mark.parametrize("max_ctas", [8, 32, 0])
@pytest.mark.parametrize("slow_consumer", [False, True])
@pytest.mark.parametrize("thr", [(1, 1), (4, 5)])
def test_overlapped_random_batches(max_ctas, slow_consumer, thr):
    """configs[1] in small (dense + sparse rows, groups of 256): a different seeded id batch per step through
    ibp_gather_decompress, strict and thresholded codecs; repeats kept so the de-duplication pre-pass and its workspace
    (stream-ordered allocations on the fetch stream) run inside the overlapped schedule too."""
    w = workloads.GNN(n_rows=40_000, batch=20_000)
    X = w.table()
    Xb = _u8(X)
    h = ibp.ibp_build(X, 512, 0, 256, align_bytes=32, threshold=thr).upload_metadata(0).set_dedup_mode(1).set_order_mode(1)
    if max_ctas:
        h.configure(max_ctas, 0)
    rng = np.random.default_rng(99)
    batches = [rng.integers(0, w.n_rows, size=20_000).astype(np.int64) for _ in range(N_STEPS)]
    ids_dev = [torch.from_numpy(b).cuda() for b in batches]

    def fetch(i, buf, stream_ptr):
        h.gather_decompress(ids_dev[i].data_ptr(), len(batches[i]), buf.data_ptr(), stream_ptr)

    got = _run(fetch, 20_000, 512, N_STEPS, slow_consumer)
    ds = oracle.Dataset(Xb, 0, 256) if thr[0] == thr[1] else oracle.DatasetT(Xb, 0, 256, thr[0], thr[1])
    for i in range(N_STEPS):
        assert np.array_equal(got[i], oracle.gather_plain(Xb, batches[i])), f"step {i}: stale or half-written buffer"
        assert np.array_equal(got[i][:512], ds.gather_decompress(batches[i][:512]))
    ds.close()
    h.destroy()


def test_overlapped_kv_spans_with_consumer_gemm():
    """configs[3] in small: page spans (index_span 512) fetched per step while the consumer runs a GEMM on the previous step's
    rows AND copies them; the GEMM result is checked against the same GEMM on the original rows (same kernel, same inputs:
    bit-identical), the copy against the plain gather."""
    w = workloads.KV(layers=2, pages=32, pages_per_layer=6)
    X = w.table()
    Xb = _u8(X)
    h = ibp.ibp_build(X, 256, 0, 16, align_bytes=16, index_span=w.index_span).upload_metadata(0).configure(16, 0)
    n = w.batch_ids
    batches = [w.ids(i) for i in range(N_STEPS)]
    ids_dev = [torch.from_numpy(b).cuda() for b in batches]
    rows = n * w.index_span
    bufs = [torch.zeros((rows, 256), dtype=torch.uint8, device="cuda") for _ in range(2)]
    results = [torch.zeros((rows, 256), dtype=torch.uint8, device="cuda") for _ in range(N_STEPS)]
    act = torch.randn((64, rows), dtype=torch.bfloat16, device="cuda")
    gemm_out = [torch.zeros((64, 128), dtype=torch.bfloat16, device="cuda") for _ in range(N_STEPS)]

    def fetch(i, bi, stream_ptr):
        h.gather_decompress(ids_dev[i].data_ptr(), n, bufs[bi].data_ptr(), stream_ptr)

    def consume(i, bi):
        torch.matmul(act, bufs[bi].view(torch.bfloat16).view(rows, 128), out=gemm_out[i])
        results[i].copy_(bufs[bi])

    DoubleBufferedPipeline(fetch, consume, N_STEPS).run_overlapped()
    torch.cuda.synchronize()
    for i in range(N_STEPS):
        want = oracle.gather_plain(Xb, batches[i], w.index_span)
        assert np.array_equal(results[i].cpu().numpy(), want), f"step {i}"
        ref = torch.matmul(act, torch.from_numpy(want).cuda().view(torch.bfloat16).view(rows, 128))
        assert torch.equal(ref.view(torch.int16), gemm_out[i].view(torch.int16)), f"step {i}: the GEMM consumed other bytes"
    h.destroy()
