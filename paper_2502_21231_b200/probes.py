"""Device ceilings the kernels are reported against, measured with the library's own probe kernels.

    python -m paper_2502_21231_b200.probes

prints, for the current CUDA device,
  * bs_reduce_probe: the rate of fp32 TMA reduce-adds (the backward's dQ reduction: 16 KB boxes of
    128 rows x 32 columns, one CTA per SM, two boxes in flight) into accumulators of growing size -
    while the accumulator's lines stay in L2, and when every line misses;
  * bs_hbm_probe: a pure-read stream and an n : 1 stream with the merge's load instruction.
bench.py reports the same figures next to the kernels' (roofline.l2_reduce, merge).  Nothing here
is on the product path; PyTorch only owns the buffers and the timing events.
"""
import json

import torch

from . import binding as B


def _time(fn, it=10):
    for _ in range(3):
        fn()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(it):
        fn()
    b.record()
    b.synchronize()
    return a.elapsed_time(b) * 1e-3 / it


def reduce_rates(rows_list=(1024, 4096, 16384, 32768), heads=32, head_dim=128, boxes=256):
    """GB/s of bs_reduce_probe on fp32 accumulators [rows][heads][head_dim]."""
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    acc = torch.zeros((max(rows_list), heads, head_dim), dtype=torch.float32, device="cuda")
    out = {}
    for rows in rows_list:
        a = acc[:rows]
        t = _time(lambda: B.reduce_probe(a, boxes))
        out[f"{rows * heads * head_dim * 4 / 2**20:.0f} MiB"] = round(n_sm * boxes * 16384 / t / 1e9, 1)
    return out


def stream_rates(n_in=8, mib_per_stream=256):
    """GB/s of bs_hbm_probe: n_in streams read and one written, and n_in + 1 streams only read."""
    n = mib_per_stream * 2**20
    ins = [torch.zeros(n, dtype=torch.uint8, device="cuda") for _ in range(n_in + 1)]
    sink = torch.zeros(4, dtype=torch.uint8, device="cuda")
    t1 = _time(lambda: B.hbm_probe(ins[:n_in], ins[n_in], sink))
    t2 = _time(lambda: B.hbm_probe(ins, None, sink))
    return {"n_to_1": round((n_in + 1) * n / t1 / 1e9, 1), "pure_read": round((n_in + 1) * n / t2 / 1e9, 1)}


if __name__ == "__main__":
    print(json.dumps({"device": torch.cuda.get_device_name(0),
                      "reduce_add_gbs_by_accumulator_size": reduce_rates(),
                      "stream_gbs": stream_rates()}))
