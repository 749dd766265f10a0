"""Prints the issue-cost microbenchmarks of libgmapp.so (gmapp_microbench, csrc/gmapp_microbench.cuh) as a markdown table:

    python -m paper_2606_12579_b200.microbench

Needs a B200; the recorded output is profiles/r02_microbench.md."""
import torch

from . import api


def main():
    assert torch.cuda.is_available(), "needs cuda:0"
    ctx = api.Context(max_agents=1, max_spheres=1)
    print("| instruction (8 independent chains, 4 warps per SM sub-partition) | SM cycles per warp-instruction per sub-partition |")
    print("|---|---|")
    for k, name in enumerate(api.MICROBENCH_KINDS):
        print(f"| {name} | {ctx.microbench(k):.2f} |")
    print(f"\nFFMA microkernel: {ctx.measure_fp32_peak(False):.1f} TFLOP/s, FFMA2: {ctx.measure_fp32_peak(True):.1f} TFLOP/s "
          f"on {ctx.sm_count} SMs ({torch.cuda.get_device_name(0)})")
    ctx.close()


if __name__ == "__main__":
    main()
