"""include/ibp.h promises: "concurrent gather/decompress calls on one handle are allowed".  Several host threads, each with its own
CUDA stream, hammer ONE handle (and one cache) with random-row gathers, span gathers, ranges and resident decodes at the same time
-- ctypes releases the GIL inside every call, so the calls really overlap -- and every result is compared with the plain gather
(oracle c1).  Also: the thread-local error text of one thread is not disturbed by another thread's successful calls.
"""
import threading

import numpy as np
import pytest

import oracle
from paper_2605_30728_b200 import binding as ibp
from paper_2605_30728_b200 import datagen

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _table(n, rb, seed):
    return (datagen.random_bytes(n * rb, seed).reshape(n, rb) & datagen.random_bytes(rb, seed + 1)[None, :]) | 0x01


@pytest.mark.parametrize("thr", [(1, 1), (4, 5)])
def test_threads_share_one_handle(thr):
    n, rb, G = 40_960, 256, 64
    X = _table(n, rb, 17)
    h = ibp.ibp_build(X, rb, 0, G, align_bytes=32, threshold=thr).upload_metadata(0)
    hs = ibp.ibp_build(X, rb, 0, G, align_bytes=16, index_span=128, threshold=thr).upload_metadata(0)   # span gathers
    cache = ibp.Cache(h, h.info().packed_bytes_stored // 3, 2)
    cache.insert(np.random.default_rng(1).permutation(n)[: n // 2])
    ptr, nbytes = h.packed_range(0, n)
    staged = torch.from_numpy(h.packed_view(ptr, nbytes).copy()).cuda()
    torch.cuda.synchronize()
    errors = []

    def worker(t):
        try:
            torch.cuda.set_device(0)
            stream = torch.cuda.Stream()
            rng = np.random.default_rng(100 + t)
            with torch.cuda.stream(stream):
                for it in range(12):
                    kind = (t + it) % 5
                    if kind == 0:                                             # random rows, large batch (pre-passes: workspaces per call)
                        ids = rng.integers(0, n, 30_000).astype(np.int64)
                        out = torch.empty((len(ids), rb), dtype=torch.uint8, device="cuda")
                        h.gather_decompress(torch.from_numpy(ids).cuda().data_ptr(), len(ids), out.data_ptr(), stream.cuda_stream)
                        want = X[ids]
                    elif kind == 1:                                           # through the cache
                        ids = rng.integers(0, n, 20_000).astype(np.int64)
                        out = torch.empty((len(ids), rb), dtype=torch.uint8, device="cuda")
                        cache.gather_decompress(torch.from_numpy(ids).cuda().data_ptr(), len(ids), out.data_ptr(), stream.cuda_stream)
                        want = X[ids]
                    elif kind == 2:                                           # spans (stream kernels)
                        ids = rng.integers(0, n // 128, 50).astype(np.int64)
                        out = torch.empty((len(ids) * 128, rb), dtype=torch.uint8, device="cuda")
                        hs.gather_decompress(torch.from_numpy(ids).cuda().data_ptr(), len(ids), out.data_ptr(), stream.cuda_stream)
                        want = oracle.gather_plain(X, ids, 128)
                    elif kind == 3:                                           # a range from the host store
                        first = int(rng.integers(0, n // G - 100)) * G
                        cnt = int(rng.integers(1, 100)) * G
                        out = torch.empty((cnt, rb), dtype=torch.uint8, device="cuda")
                        h.gather_decompress_range(first, cnt, out.data_ptr(), stream.cuda_stream)
                        want = X[first:first + cnt]
                    else:                                                     # resident decode of the staged table
                        out = torch.empty((n, rb), dtype=torch.uint8, device="cuda")
                        h.decompress_resident(staged.data_ptr(), 0, n, out.data_ptr(), stream.cuda_stream)
                        want = X
                    stream.synchronize()
                    if not np.array_equal(out.cpu().numpy(), want):
                        errors.append(f"thread {t} iteration {it} kind {kind}: wrong bytes")
                # a failing call in THIS thread: its error text is this thread's own
                try:
                    h.gather_decompress_range(1, 5, out.data_ptr(), stream.cuda_stream) if thr == (1, 1) else h.gather_decompress_range(0, n + 1, out.data_ptr(), stream.cuda_stream)
                    errors.append(f"thread {t}: the bad range was accepted")
                except ibp.IbpError as e:
                    if "range" not in str(e) and "unit" not in str(e) and "first_row" not in str(e):
                        errors.append(f"thread {t}: unexpected error text {e}")
        except Exception as e:                                                # noqa: BLE001 -- reported through the list
            errors.append(f"thread {t}: {type(e).__name__}: {e}")

    threads = [threading.Thread(target=worker, args=(t,)) for t in range(6)]
    for th in threads:
        th.start()
    for th in threads:
        th.join(timeout=300)
    assert not any(th.is_alive() for th in threads), "a worker hung"
    assert not errors, errors
    cache.destroy(); h.destroy(); hs.destroy()
