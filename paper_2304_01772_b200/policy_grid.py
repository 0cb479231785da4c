"""Measure the kernel-selection policies of the int8 Ising path on a (batch, L) grid: flips/ns of SPIN_POLICY_AUTO,
STREAMING, RESIDENT, PERSISTENT and TILED (CUDA-event timing through the binding, best of 3).  Prints a markdown table; the
crossovers it shows are what `use_resident` / `use_persistent` in csrc/spin_api.cu encode (profiles/r2_policy_grid.md).

    python -m paper_2304_01772_b200.policy_grid
"""
import sys

import numpy as np


def main():
    import torch

    import paper_2304_01772_b200 as sp
    names = {sp.SPIN_POLICY_AUTO: "auto", sp.SPIN_POLICY_STREAMING: "streaming", sp.SPIN_POLICY_RESIDENT: "resident",
             sp.SPIN_POLICY_PERSISTENT: "persistent", sp.SPIN_POLICY_TILED: "tiled"}
    stream = torch.cuda.Stream()
    print("| batch | L | sites | auto picks | auto | streaming | resident | persistent | tiled |")
    print("|---|---|---|---|---|---|---|---|---|")
    for L in (64, 128, 224, 256, 416, 640, 1024, 2560):
        for batch in (1, 4, 16, 64, 256):
            sites = batch * L * L
            if sites > (1 << 27):
                continue
            n = int(max(20, min(2000, 4e9 / sites / 4)))
            row = []
            picked = ""
            for policy in (sp.SPIN_POLICY_AUTO, sp.SPIN_POLICY_STREAMING, sp.SPIN_POLICY_RESIDENT, sp.SPIN_POLICY_PERSISTENT,
                           sp.SPIN_POLICY_TILED):
                sim = sp.spin_create_ex(batch, L, sp.SPIN_MODEL_ISING, seed=1, cuda_stream=stream.cuda_stream)
                sim.spin_set_policy(policy)
                variant = sim.spin_kernel_variant()
                if policy == sp.SPIN_POLICY_AUTO:
                    picked = variant.replace("ising_int8_", "")
                elif names[policy] not in variant and policy != sp.SPIN_POLICY_STREAMING:
                    row.append("-")                      # the shape does not qualify: the call would stream
                    sim.spin_destroy()
                    continue
                beta = np.full(batch, 0.44)
                sim.spin_sweep(beta, 1.0, 0.0, n, 0)
                sim.spin_synchronize()
                best = 0.0
                for rep in range(3):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    sim.spin_sweep(beta, 1.0, 0.0, n, (rep + 1) * n)
                    e1.record(stream)
                    sim.spin_synchronize()
                    best = max(best, sites * n / (e0.elapsed_time(e1) * 1e6))
                row.append("%.1f" % best)
                sim.spin_destroy()
            print("| %d | %d | %d | %s | %s |" % (batch, L, sites, picked, " | ".join(row)), flush=True)


if __name__ == "__main__":
    sys.exit(main())
