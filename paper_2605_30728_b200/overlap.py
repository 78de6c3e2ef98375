"""S7: stream-overlap harness -- batch i+1's fetch+decode against a consumer kernel on batch i.

    fetch stream   : step i+1 -> ibp gather/decode into buffer (i+1) % 2
    consumer stream: step i   -> consumer kernel(s) reading buffer i % 2           ("We reserved only 64
                                                                                    SMs for decompression")
Events order the two streams: the consumer of step i waits for fetched[i]; the fetch of step i+2 waits for
consumed[i] before it overwrites the buffer.  The decode kernels are persistent with a bounded grid
(`ibp_configure(max_ctas)`), so the SM share of the fetch is a launch parameter, not a side effect.

Only stream/event plumbing lives here (torch supplies streams and events); every byte is moved by the library's kernels
and by whatever consumer the caller passes in.
"""
from __future__ import annotations

import torch


class DoubleBufferedPipeline:
    """fetch(i, buffer_index, cuda_stream_ptr) and consume(i, buffer_index) are callables; n_steps steps."""

    def __init__(self, fetch, consume, n_steps: int, device=None, fetch_priority_high: bool = True):
        self.fetch, self.consume, self.n = fetch, consume, n_steps
        lo, hi = torch.cuda.Stream.priority_range() if hasattr(torch.cuda.Stream, "priority_range") else (0, -1)
        self.s_fetch = torch.cuda.Stream(device=device, priority=hi if fetch_priority_high else lo)
        self.s_cons = torch.cuda.Stream(device=device, priority=lo)

    # ---- reference schedules, all timed with CUDA events on the streams they use -------------------------------
    def run_fetch_only(self):
        with torch.cuda.stream(self.s_fetch):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for i in range(self.n):
                self.fetch(i, i % 2, self.s_fetch.cuda_stream)
            b.record()
        b.synchronize()
        return a.elapsed_time(b)

    def run_consume_only(self):
        with torch.cuda.stream(self.s_cons):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for i in range(self.n):
                self.consume(i, i % 2)
            b.record()
        b.synchronize()
        return a.elapsed_time(b)

    def run_serial(self):
        """fetch(i) then consume(i) on one stream: what a blocking copy-then-compute loop costs."""
        with torch.cuda.stream(self.s_cons):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for i in range(self.n):
                self.fetch(i, i % 2, self.s_cons.cuda_stream)
                self.consume(i, i % 2)
            b.record()
        b.synchronize()
        return a.elapsed_time(b)

    def run_overlapped(self):
        """fetch(i+1) on the fetch stream while consume(i) runs on the consumer stream; two buffers."""
        fetched = [torch.cuda.Event() for _ in range(self.n)]
        consumed = [torch.cuda.Event() for _ in range(self.n)]
        start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        start.record(self.s_fetch)
        self.s_cons.wait_event(start)
        for i in range(self.n):
            if i >= 2:
                self.s_fetch.wait_event(consumed[i - 2])          # buffer i % 2 is free again
            with torch.cuda.stream(self.s_fetch):
                self.fetch(i, i % 2, self.s_fetch.cuda_stream)
                fetched[i].record(self.s_fetch)
            self.s_cons.wait_event(fetched[i])
            with torch.cuda.stream(self.s_cons):
                self.consume(i, i % 2)
                consumed[i].record(self.s_cons)
        self.s_fetch.wait_event(consumed[self.n - 1])
        stop.record(self.s_fetch)
        stop.synchronize()
        return start.elapsed_time(stop)


def summarize(t_fetch, t_consume, t_serial, t_overlap):
    ideal = max(t_fetch, t_consume)
    hidden = t_serial - t_overlap
    return {
        "fetch_only_ms": round(t_fetch, 3), "consume_only_ms": round(t_consume, 3), "serial_ms": round(t_serial, 3),
        "overlapped_ms": round(t_overlap, 3), "ideal_ms": round(ideal, 3),
        "overlap_efficiency": round(ideal / t_overlap, 4) if t_overlap > 0 else None,   # 1.0 = the shorter leg is fully hidden
        "hidden_ms": round(hidden, 3),
    }
