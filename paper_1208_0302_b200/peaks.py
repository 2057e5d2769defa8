"""Measures the ALU roofline denominators on the box (SURVEY.md par. 8(d): MEASURED_PEAKS.json has no FP32 / SFU peak).

`python -m paper_1208_0302_b200.peaks` prints one JSON object: lane-slots/s of each probe of include/me.h's
me_peak_probe (FFMA, FFMA2, MUFU), the flop/s they imply, and the SM clock sampled during the run.
Argument marshalling and CUDA-event timing only; the probes are kernels of libme_b200.so.
"""
import json

KINDS = {0: ("ffma", 1, 0, 0), 1: ("ffma2", 0, 1, 0), 3: ("mufu", 0, 0, 1)}
FLOP_PER_SLOT = {0: 2.0, 1: 4.0, 3: 0.0}


def measure(iters=4096, blocks_per_sm=8, repeats=5, kinds=None):
    import torch
    from . import binding as B
    B.lib()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    blocks = sms * blocks_per_sm
    scratch = torch.zeros(blocks * 256, dtype=torch.float32, device="cuda")
    out = {"sm_count": sms, "iters": iters, "blocks": blocks, "probes": {}}
    for kind, (name, n_ffma, n_ffma2, n_mufu) in KINDS.items():
        if kinds is not None and kind not in kinds:
            continue
        B.me_peak_probe(kind, 64, blocks, scratch)
        torch.cuda.synchronize()
        best = None
        for _ in range(repeats):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            slots = B.me_peak_probe(kind, iters, blocks, scratch)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best = ms if best is None else min(best, ms)
        sec = best * 1e-3
        out["probes"][name] = {"ms": best, "slots_per_s": slots / sec,
                               "thread_inst_per_s": slots * (n_ffma + n_ffma2 + n_mufu) / sec,
                               "tflops": slots * FLOP_PER_SLOT[kind] / sec / 1e12,
                               "per_sm_per_clk_at_1965MHz": slots * (n_ffma + n_ffma2 + n_mufu) / sec / sms / 1.965e9}
    return out


if __name__ == "__main__":
    print(json.dumps(measure(), indent=1))
