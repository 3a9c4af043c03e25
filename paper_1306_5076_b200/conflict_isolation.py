"""The bank-conflict isolation experiment (profiles/r3_conflict_isolation.md).

    python -m paper_1306_5076_b200.conflict_isolation [--log2n 24]

Runs, on the same seeded uint32 input, the production kernels and their phase-separated variants
(include/bcf.h, bcf_debug_*_isolated) so that one `ncu --metrics l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_ld.sum,
l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_st.sum,...` pass over this script lists, kernel by kernel:
  tile_mergesort_kernel                      production, several CTAs per SM, loads / sorts / stores overlap
  tile_mergesort_isolated_kernel  (grid A)   phases separated by barriers, ONE CTA per SM        -> expected 0
  tile_mergesort_isolated_kernel  (grid B)   same code, several CTAs per SM (phases of different CTAs overlap)
  merge_pipe_kernel                          production, TMA producer + consumers + stores overlap
  merge_round_isolated_kernel     (grid A)   phases separated, ONE CTA per SM                    -> expected 0
  merge_round_isolated_kernel     (grid B)   the same launch again: the experiment has the production shape (16-page
                                             shares, 16 warps, one CTA per SM is all that fits), `exclusive` changes nothing
Every output is checked against the production result before the script exits (exit code 1 on a mismatch).
Launch order = the order above; the isolated kernels appear twice in ncu's list, exclusive (A) first.
"""
import argparse
import sys

import numpy as np
import torch

import paper_1306_5076_b200 as bcf
from paper_1306_5076_b200 import workloads


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--log2n", type=int, default=24, help="keys (2^24: 16384 tiles / 2048 shares, many waves on 148 SMs)")
    args = ap.parse_args()
    n = 1 << args.log2n
    keys = workloads.cfg3_sort_u32(n=n)
    src = torch.from_numpy(keys.view(np.int32)).cuda()

    # ---- tile sorts
    want = src.clone()
    bcf.sort_tiles_mergesort(want)
    for exclusive in (True, False):
        got = src.clone()
        bcf.debug_sort_tiles_isolated(got, exclusive=exclusive)
        torch.cuda.synchronize()
        if not torch.equal(got, want):
            print("tile sort mismatch, exclusive =", exclusive)
            return 1

    # ---- one merge round: two sorted runs of n / 2
    runs = torch.from_numpy(workloads.sorted_runs(keys, n // 2).view(np.int32)).cuda()
    want = bcf.merge_runs(runs, n // 2)
    for exclusive in (True, False):
        got = bcf.debug_merge_round_isolated(runs, n // 2, exclusive=exclusive)
        torch.cuda.synchronize()
        if not torch.equal(got, want):
            print("merge round mismatch, exclusive =", exclusive)
            return 1
    print("conflict_isolation: all variants equal the production kernels on 2^%d keys" % args.log2n)
    return 0


if __name__ == "__main__":
    sys.exit(main())
