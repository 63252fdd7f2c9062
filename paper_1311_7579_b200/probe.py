"""Issue-cost table of the fp64 instruction patterns the kernels are made of (profiles/r2_dfma_issue.md).

    python -m paper_1311_7579_b200.probe            # CUDA events + SM clock -> cycles per warp instruction and sub-partition

Every row is one launch of ``osc_fp64_issue_probe`` (8 warps per sub-partition, 8 independent chains per thread), timed
with CUDA events; cycles = time x clocks.sm, per sub-partition: 8 warps x 8 chains x iters x (instructions per chain
step) warp instructions.  The same launches under ncu (smsp__inst_executed.sum, sm__cycles_elapsed.max) give the
figures without the clock assumption.  Measurement only: nothing of the method is computed here.
"""
from __future__ import annotations


KINDS = [(0, "DFMA x = fma(y, z, x): three distinct register operands", 1),
         (1, "DFMA x = fma(x, y, imm): two registers", 1),
         (2, "DFMA x = fma(x, imm, imm): one register", 1),
         (3, "DMUL x = x * y", 1),
         (4, "DADD x = x + y", 1),
         (5, "DFMA (three registers) + 2 FFMA (three registers each)", 3),
         (6, "DFMA (three registers) + 2 IMAD", 3)]


def sm_clock_mhz() -> float:
    """Current SM clock through NVML (a call of microseconds: usable while the probe launches are running)."""
    import pynvml

    pynvml.nvmlInit()
    return float(pynvml.nvmlDeviceGetClockInfo(pynvml.nvmlDeviceGetHandleByIndex(0), pynvml.NVML_CLOCK_SM))


def main(iters: int = 1 << 14) -> None:
    import torch

    from . import binding as osc

    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    osc.osc_set_device(0)
    print("| kind | pattern | us per launch | SM MHz during launch | cycles per pattern | cycles per warp instruction |")
    print("|---|---|---|---|---|---|")
    for kind, what, n_inst in KINDS:
        for _ in range(2):
            osc.osc_fp64_issue_probe(kind, iters, 4)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record()
        for _ in range(20):
            osc.osc_fp64_issue_probe(kind, iters, 4)
        b.record()
        mhz = sm_clock_mhz()                                  # sampled while the launches run (20 x ~2 ms)
        torch.cuda.synchronize()
        us = 1e3 * a.elapsed_time(b) / 20
        per_pattern = us * mhz / (8 * 8 * iters)              # 8 warps per sub-partition x 8 chains per thread
        print(f"| {kind} | {what} | {us:.1f} | {mhz:.0f} | {per_pattern:.2f} | {per_pattern / n_inst:.2f} |")


if __name__ == "__main__":
    main()
