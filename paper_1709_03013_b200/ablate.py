"""Timing ablations of the fp4 tensor kernel (developer aid; profiles/r1f… and r1g… quote its output).

    python -m paper_1709_03013_b200.ablate --config 2 --debug 0,14,9,63,64

The script builds and loads libcsg_ablate.so -- the library's sources compiled with -DCSG_ABLATE, which adds the
ablation switches to the fp4 instantiation of tensor_action_kernel and exports csg_set_debug -- INSTEAD of libcsg.so
(the product library has neither).  For every value of --debug it calls csg_set_debug (bits: 1 no MMA issue, 2 no expansion arithmetic, 4 no
operand stores, 8 no bucketing in the epilogue, 16 no fence before publishing a stage, 32 no packed-bit ring, 64 free-running
producers, 128 no prefill before the epilogue, 256 no open-range masks; any non-zero value gives WRONG counts), and the
CUDA-event time of the interval kernel (csg_last_kernel_ms) of four calls is printed.  Needs a B200.
"""
import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    import ctypes
    import torch
    import csg_inputs
    import paper_1709_03013_b200 as csg
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2, help="index into csg_inputs.CONFIGS")
    ap.add_argument("--debug", default="0,14,9,63,64", help="comma-separated CSG_DEBUG values")
    ap.add_argument("--runs", type=int, default=4)
    ap.add_argument("--sparse", type=int, default=0, help="csg_set_sparse mode: 0 auto, 1 on, 2 off (dense sweep)")
    args = ap.parse_args()
    csg.LIB_PATH = csg._build.build(ablate=True)       # never the product library
    lib = csg.load()
    lib.csg_set_debug.argtypes = [ctypes.c_int]
    cfg = csg_inputs.CONFIGS[args.config]
    N, dim = cfg["N"], cfg["dim"]
    _, bits = csg_inputs.make_config(cfg)
    d = csg.to_device(bits)
    csg.csg_set_variant(csg.VARIANT_TENSOR_FP4)
    csg.csg_set_sparse(args.sparse)
    csg.csg_set_kernel_timing(True)
    for dbg in [int(x) for x in args.debug.split(",")]:
        lib.csg_set_debug(dbg)
        ms = []
        for _ in range(args.runs):
            csg.csg_action(d, N, dim, 1.0, 3)
            torch.cuda.synchronize()
            ms.append(csg.csg_last_kernel_ms())
        print("%s sparse=%d CSG_DEBUG=%-4d kernel ms %s" % (cfg["name"], args.sparse, dbg, " ".join("%.3f" % m for m in ms)), flush=True)
    lib.csg_set_debug(0)
    csg.csg_set_kernel_timing(False)
    csg.csg_set_variant(csg.VARIANT_AUTO)


if __name__ == "__main__":
    main()
