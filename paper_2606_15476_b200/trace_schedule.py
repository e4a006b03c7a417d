"""Device-timer trace of the per-call schedule on configs[4] (development tool; evidence for DESIGN.md sections 14-15).

    python -m paper_2606_15476_b200.build --trace          # libfarm_trace.so: the library with -DFARM_TRACE
    python -m paper_2606_15476_b200.trace_schedule [--inputs-ready 0|1] [--calls 14]

The trace build stamps %globaltimer (and clock64 of CTA 0) inside the similarity, association and merge kernels, one row per
call.  This script integrates back-to-back 16-frame batches of the stress scene and prints, per call and relative to the start
of its similarity kernel: when the kernel's last CTA started, when the prep share and the waits were over, when the kernel
ended, where the previous call's decision scan and merge fell, and the SM clock over the kernel's lifetime.  Numbers under a
trace build are not bench values.
"""
import argparse
import ctypes as C
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2606_15476_b200 import binding  # noqa: E402


def single_frame(opt, binding):
    """single-frame calls of configs 1-3 with the split schedule: where the time of a call goes"""
    from paper_2606_15476_b200 import FarmMap, scenes as S
    cfg = S.get_config(opt.config)
    n = opt.calls
    frames = S.generate_frames(opt.config, range(20, 20 + n))
    dev = torch.device("cuda", 0)
    stream = torch.cuda.Stream(device=dev)
    m = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype, stream=stream.cuda_stream,
                max_objects=8192, max_voxels=1 << 24, max_det_per_call=64, inputs_ready=opt.inputs_ready)
    staged = []
    with torch.cuda.stream(stream):
        for fr in frames:
            desc = np.ascontiguousarray(fr.desc).view(np.int16)
            staged.append((torch.from_numpy(fr.depth).to(dev), torch.from_numpy(fr.mask.view(np.int16)).to(dev),
                           torch.from_numpy(np.ascontiguousarray(fr.K, np.float32)).to(dev),
                           torch.from_numpy(np.ascontiguousarray(fr.T, np.float32)).to(dev), torch.from_numpy(desc).to(dev), fr.n_det))
    torch.cuda.synchronize()
    lib = binding.load_library()
    names = ("sim", "assoc", "lift", "probe")
    for name in names:
        getattr(lib, f"farm_trace_{name}_read")(None, 1)
    for d in staged:
        m.integrate(*d)
    m.sync()
    t = {}
    for name in names:
        x = np.zeros((16, 8), np.uint64)
        getattr(lib, f"farm_trace_{name}_read")(x.ctypes.data_as(C.c_void_p), 0)
        t[name] = x.astype(np.int64)
    print(f"configs[{opt.config}], {n} single-frame calls back to back, FARM_OPT_INPUTS_READY = {opt.inputs_ready}; us relative to the end of the"
          " previous call's merge warps")
    print("call | prep start | lift start / end | similarity start / end | probe start / end | scoring start / over | scan start / end |"
          " merge start / warps end | period")
    print("probe kernel, us after its first CTA passed the wait: first CTA resident | last warp with records past its record loads |"
          " the block hash | the pair set | phase B | last CTA end")
    for c in range(n - 7, n + 1):
        l, p = t["lift"][c & 15], t["probe"][c & 15]
        g = lambda x: f"{(x - l[2]) / 1e3:6.1f}"
        print(f"{c:4d} | {g(p[0])} | {g(p[1])} | {g(p[3])} | {g(p[5])} | {g(p[7])} | {g(l[3])}")
    for c in range(n - 7, n + 1):
        s, a, l = t["sim"][c & 15], t["assoc"][c & 15], t["lift"][c & 15]
        t0 = t["assoc"][(c - 1) & 15][7]
        f = lambda x: f"{(x - t0) / 1e3:6.1f}"
        print(f"{c:4d} | {f(l[4])} | {f(l[0])} / {f(l[1])} | {f(s[0])} / {f(s[7])} | {f(l[2])} / {f(l[3])} | {f(a[0])} / {f(a[1])} | {f(a[3])} / {f(a[5])} | "
              f"{f(a[2])} / {f(a[7])} | {(a[7] - t0) / 1e3:6.1f}")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--inputs-ready", type=int, default=1)
    ap.add_argument("--calls", type=int, default=14)
    ap.add_argument("--config", type=int, default=4, help="4: 16-frame stress batches; 1-3: single-frame calls of that config")
    opt = ap.parse_args()
    lib_path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libfarm_trace.so")
    if not os.path.exists(lib_path):
        raise SystemExit("build the trace library first: python -m paper_2606_15476_b200.build --trace")
    binding.LIB_PATH = lib_path
    sys.argv = sys.argv[:1]
    import bench  # the stress scene and its import arrays (repo root)
    from paper_2606_15476_b200 import FarmMap, scenes as S

    if opt.config != 4:
        return single_frame(opt, binding)
    args = bench.parse()
    args.steps, args.warmup, args.extra_batches = opt.calls, 0, 0
    dev = torch.device("cuda", 0)
    stream = torch.cuda.Stream(device=dev)
    cfg = S.get_config(4)
    sc, keys, owner, n_vox, desc = bench.build_stress(args)
    objs = bench.object_records(binding.OBJECT_DTYPE, n_vox)
    m = FarmMap(cfg.voxel, cfg.D, cfg.w_geo, cfg.w_sem, cfg.tau, H=cfg.H, W=cfg.W, dtype=cfg.dtype, max_objects=len(objs) + 40000,
                max_voxels=int(len(keys) * 1.05) + 20 * 600000, max_blocks=len(keys) // 16 + 20 * 20000, max_det_per_call=1600,
                max_frames_per_call=16, max_pairs_per_call=1 << 21, stream=stream.cuda_stream, inputs_ready=opt.inputs_ready)
    m.import_(objs, desc, keys, owner)
    batches = []
    for b in range(opt.calls):
        depth, mask, K, T, dsc, n_det = bench.batch_host_arrays(sc.batch(b))
        batches.append((torch.from_numpy(depth).to(dev), torch.from_numpy(mask.view(np.int16)).to(dev), torch.from_numpy(K).to(dev),
                        torch.from_numpy(T).to(dev), torch.from_numpy(dsc.view(np.int16)).to(dev), n_det))
    torch.cuda.synchronize()
    lib = binding.load_library()
    tables = {}
    for name in ("sim", "assoc", "tiles", "clock", "lift"):
        getattr(lib, f"farm_trace_{name}_read")(None, 1)
    for b in range(opt.calls):
        m.integrate_batch(16, *batches[b])
    m.sync()
    for name in ("sim", "assoc", "tiles", "clock"):
        t = np.zeros((16, 8), np.uint64)
        getattr(lib, f"farm_trace_{name}_read")(t.ctypes.data_as(C.c_void_p), 0)
        tables[name] = t.astype(np.int64)
    split = opt.inputs_ready == 1
    print(f"configs[4], {opt.calls} calls back to back, FARM_OPT_INPUTS_READY = {opt.inputs_ready}"
          f" ({'split schedule from call 3 on' if split else 'stream-ordered schedule'}); times in us")
    if not split:
        # without the option every call writes row 0 of the tables: the last call
        c = tables["clock"][0]
        print(f"last call: CTA 0 of the similarity kernel lived {c[1] / 1e3:.1f} us at {c[0] / max(c[1], 1) * 1e3:.0f} MHz")
        a = tables["assoc"][0]
        print(f"last call: decision scan {(a[5] - a[3]) / 1e3:.1f} us, merge warps done {(a[7] - a[5]) / 1e3:.1f} us after the scan")
        return
    print("call | last CTA start | prep share done (first / last) | first phase-2 tile | end | prev scan (start / end) | prev merge (start / end) |"
          " phase-2 epilogues done (first / last) | CTA 0 lifetime | SM MHz")
    for c in range(max(4, opt.calls - 8), opt.calls + 1):
        s, a, tt, ck = tables["sim"][c & 15], tables["assoc"][(c - 1) & 15], tables["tiles"][c & 15], tables["clock"][c & 15]
        t0 = s[0]
        f = lambda x: f"{(x - t0) / 1e3:6.1f}"
        print(f"{c:4d} | {f(s[1])} | {f(s[6])} / {f(s[3])} | {f(s[2])} | {f(s[7])} | {f(a[3])} / {f(a[5])} | {f(a[2])} / {f(a[7])} | "
              f"{f(tt[4])} / {f(tt[5])} | {ck[1] / 1e3:6.1f} | {ck[0] / max(ck[1], 1) * 1e3:5.0f}")


if __name__ == "__main__":
    main()
