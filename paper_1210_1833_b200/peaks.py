"""Print the measured unit throughputs of this GPU (cute_measure_peaks) as a Markdown table.

    python -m paper_1210_1833_b200.peaks

These are the denominators of the pair kernel's roofline; bench.py calls the same
entry point in every run.
"""
from __future__ import annotations

import sys


def main() -> int:
    import torch
    from . import api
    peaks = api.cute_measure_peaks()
    prop = torch.cuda.get_device_properties(0)
    print(f"device: {prop.name}, {prop.multi_processor_count} SMs; one 512-thread CTA per SM, clock64() timing\n")
    print("| instruction (or mix) | lane-ops / clk / SM | warp-instr / clk / SM |")
    print("|---|---|---|")
    for name, (ops, ins) in peaks.items():
        print(f"| {name} | {ops:.1f} | {ins:.2f} |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
