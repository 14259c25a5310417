#!/usr/bin/env python
"""bench.py -- one-line JSON benchmark of the HASTE hot path on B200.

A step = one pass of the whole hot path over one synthetic batch of BASELINE.json config 3
(670K labels: B=512, d=768, tail 653 707 labels G=64 K=128, dense head 16 384 labels, bf16):
  haste_forward_loss + haste_backward (sparse tail) + haste_head_forward_loss + haste_head_backward.
`value` = algorithmic TFLOP/s of the step (2*B*L_t*K per tail pass x3 + 2*B*L_h*d per head pass x3),
inputs resident in HBM; `e2e` = the same with the step's inputs (X, X_head, CSR targets) copied from
pinned host memory and the step's results (losses, dX, dX_head) copied back, every step.
`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
Multi-GPU: the path does not shard ("replicas only"): N ranks run N independent replicas.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

WORKLOAD = "670k"


def _flops(cfg):
    tail = 2.0 * cfg.B * cfg.L_t * cfg.K
    head = 2.0 * cfg.B * cfg.L_h * cfg.d
    return tail, head


def _alg_bytes(cfg, dw_bytes=None):
    """Algorithmic HBM bytes per launch of each tail kernel."""
    e = 2 if cfg.dtype == "bf16" else 4          # element size of X, W, dY (and dW unless stated)
    dw_bytes = e if dw_bytes is None else dw_bytes
    W = cfg.L_t * cfg.K * e
    idx = cfg.NG * cfg.K * 4
    dY = cfg.NG * cfg.G * cfg.B * e
    X = cfg.B * cfg.d * e
    dX = cfg.B * cfg.d * 4
    return {
        "forward": W + idx + X + dY,
        "dW": dY + idx + X + cfg.L_t * cfg.K * dw_bytes + cfg.L_t * 4,
        "dX": dY + W + idx + dX,
        # forward + dW in one kernel (haste_forward_loss_dw): dY is written and never read back, X is gathered once
        "forward_dW": W + idx + X + dY + cfg.L_t * cfg.K * dw_bytes + cfg.L_t * 4,
    }


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        m = json.load(open(p))
        return dict(hbm=float(m["hbm_gbs"]), bf16=float(m["bf16_tflops"]), bf16_sustained=float(m.get("bf16_tflops_sustained", m["bf16_tflops"])), source="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region: an NVML polling thread (a sample every
    ~8 ms; the default --steps makes the timed region ~35 ms), `nvidia-smi -lms` as the fallback."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
    BITS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.f = None
        self.thread = None
        self.stop_flag = False
        self.rows = []      # (sm_mhz, max_mhz, watts, reason_mask)

    def _nvml_loop(self, nv, h):
        reasons_fn = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or getattr(nv, "nvmlDeviceGetCurrentClocksThrottleReasons")
        smax = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
        # NVML queries are not free for the GPU: polling every 2 ms slowed every kernel by ~7 % (measured), so poll
        # every 8 ms (~1 %), clock and reasons only; power is read once per ~8 polls
        n, watts = 0, 0.0
        while not self.stop_flag:
            try:
                if n % 8 == 0:
                    watts = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
                self.rows.append((nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM), smax, watts, int(reasons_fn(h))))
            except Exception:
                pass
            n += 1
            time.sleep(0.008)

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            # NVML enumerates physical devices: map through CUDA_VISIBLE_DEVICES when it is a plain index list
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            phys = self.index
            if vis and all(t.strip().isdigit() for t in vis.split(",")):
                phys = int(vis.split(",")[self.index])
            h = nv.nvmlDeviceGetHandleByIndex(phys)
            self.thread = threading.Thread(target=self._nvml_loop, args=(nv, h), daemon=True)
            self.thread.start()
            return
        except Exception:
            self.thread = None
        try:
            self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.thread is not None:
            self.stop_flag = True
            self.thread.join(timeout=2)
            if self.rows:
                mask = 0
                for r in self.rows:
                    mask |= r[3]
                out = {"sm_mhz": float(np.median([r[0] for r in self.rows])), "sm_max_mhz": float(max(r[1] for r in self.rows)),
                       "power_w_max": float(max(r[2] for r in self.rows)), "samples": len(self.rows),
                       "reasons": sorted(n for b, n in self.BITS.items() if mask & b), "source": "nvml"}
            return out
        if not self.proc:
            return out
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                   "samples": len(sm), "reasons": sorted(reasons), "source": "nvidia-smi"}
        return out


def _sample_inputs(cfg, n_groups):
    """A bounded sample of the workload for the CPU oracle: the first n_groups groups of the tail
    (same B, d, G, K, same generators) and the first 64*n_groups/4 head labels."""
    from paper_2606_01117_b200 import synth
    import dataclasses
    Lt = n_groups * cfg.G
    Lh = max(16, min(cfg.L_h, n_groups * 4))
    small = dataclasses.replace(cfg, L=Lt + Lh, L_h=Lh)
    return small, synth.make_inputs(small, with_head=True)


def _oracle_step(oracle, small, inp):
    r = oracle.tail_forward(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, small.G, label_offset=small.L_h, want_z=False)
    oracle.tail_backward(inp.X, inp.idx, inp.W, r["dY"], small.G)
    h = oracle.head_forward(inp.X_head, inp.W_head, None, inp.rowptr, inp.col, want_z=False)
    oracle.head_backward(inp.X_head, inp.W_head, h["dY"])


def cpu_baseline(cfg, target_s=12.0):
    """The oracle as it stands, one thread, on a bounded sample sized to about target_s seconds."""
    import oracle
    small, inp = _sample_inputs(cfg, 4)
    t0 = time.perf_counter()
    _oracle_step(oracle, small, inp)
    t1 = time.perf_counter() - t0
    ng = int(max(4, min(cfg.NG, 4 * target_s / max(t1, 1e-3))))
    small, inp = _sample_inputs(cfg, ng)
    t0 = time.perf_counter()
    _oracle_step(oracle, small, inp)
    dt = time.perf_counter() - t0
    tail, head = _flops(small)
    fl = 3 * (tail + head)
    return {"value": fl / dt / 1e12, "unit": "TFLOP/s", "cores": 1, "kind": "oracle",
            "sample": "first %d of %d tail groups (%d labels) + %d head labels of config 3, B=%d, one fwd+bwd pass, %.1f s"
                      % (ng, cfg.NG, small.L_t, small.L_h, cfg.B, dt)}


def run_reference(args, cfg):
    """--impl reference: the fp64 oracle, one thread, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    ng = 8
    small, inp = _sample_inputs(cfg, ng)
    for _ in range(args.warmup):
        _oracle_step(oracle, small, inp)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _oracle_step(oracle, small, inp)
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    tail, head = _flops(small)
    v = 3 * (tail + head) / dt / 1e12
    sample = "each step: first %d of %d tail groups (%d labels) + %d head labels of config 3 at B=%d" % (ng, cfg.NG, small.L_t, small.L_h, cfg.B)
    print(json.dumps({
        "impl": "reference", "metric": "sparse_layer_fwd_bwd_tflops_670k", "value": v, "unit": "TFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config3_670k_sample", "sample": sample},
        "cpu_baseline": {"value": v, "unit": "TFLOP/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def max_over_ranks(ms, dist, device):
    """Device time of the slowest rank (the job is as fast as its slowest replica).  `dist` is torch.distributed (any
    backend: nccl on the GPU box, gloo in the CPU tests) or None for a single process."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([float(ms)], device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_tflops(world, step_flops, ms_per_step):
    """`value`: N independent replicas ("replicas only") each do step_flops per step; weak scaling."""
    return world * step_flops / (ms_per_step * 1e-3) / 1e12


def run_sweep(args):
    """--sweep: BASELINE.json config 5 (kernel sweep at fixed nnz): B in {64,256,1024}, d=768, L=670091, K=64,
    G in {1,8,16,32,64,128} (G=1 = ungrouped per-label fixed fan-in, the comparison kernel), uniform sorted idx, no head,
    against the FLOPs-matched dense bottleneck d -> r=64 -> L in bf16 (cuBLAS through torch.matmul: comparison point,
    not product).  Timing only (parity for config 5 lives in tests/test_gpu_configs.py); inputs are drawn on the
    device with torch's generator (seed 1005).  One JSON line per point on stdout."""
    import torch
    from paper_2606_01117_b200 import haste
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    peaks = _peaks()
    d, L, K, r = 768, 670091, 64, 64
    gen = torch.Generator(device=dev)
    gen.manual_seed(1005)
    W = (torch.randn(L, K, device=dev, generator=gen) * 0.02).to(torch.bfloat16)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > L2: written between timed iterations
    Bs = [int(x) for x in args.sweep_B.split(",")]
    Gs = [int(x) for x in args.sweep_G.split(",")]
    steps = min(args.steps, 10)
    for B in Bs:
        X = torch.randn(B, d, device=dev, generator=gen).to(torch.bfloat16)
        rowptr = torch.arange(0, 5 * (B + 1), 5, dtype=torch.int32, device=dev)
        col = torch.sort(torch.randint(0, L, (B, 5), device=dev, generator=gen, dtype=torch.int32), dim=1).values.reshape(-1).contiguous()
        # dense bottleneck d -> r -> L: H = X P^T [B,r]; Z = H W^T [B,L]; backward dW = dZ^T H, dH = dZ W  (same FLOPs and W/output bytes)
        P = (torch.randn(r, d, device=dev, generator=gen) * 0.02).to(torch.bfloat16)
        Hh = X @ P.t()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        tb = {"fwd": [], "dW": [], "dX": []}
        Z = torch.empty(B, L, dtype=torch.bfloat16, device=dev)
        for it in range(steps + 2):
            flush.fill_(it & 1)
            ev[0].record(); torch.matmul(Hh, W.t(), out=Z); ev[1].record()
            dWd = Z.t() @ Hh; ev[2].record()
            dH = Z @ W; ev[3].record()
            torch.cuda.synchronize()
            if it >= 2:
                tb["fwd"].append(ev[0].elapsed_time(ev[1])); tb["dW"].append(ev[1].elapsed_time(ev[2])); tb["dX"].append(ev[2].elapsed_time(ev[3]))
        del Z, dWd, dH
        dense = {k: float(np.median(v)) for k, v in tb.items()}
        for G in Gs:
            NG = -(-L // G)
            idx = torch.empty(NG, K, dtype=torch.int32, device=dev)
            for a in range(0, NG, 65536):       # K distinct features per group, uniform, sorted
                b = min(NG, a + 65536)
                idx[a:b] = torch.sort(torch.rand(b - a, d, device=dev, generator=gen).topk(K, dim=1).indices, dim=1).values.to(torch.int32)
            layer = haste.HasteLayer(d, L, G, K, B, "bf16", flags=haste.HASTE_IDX_SORTED_DISTINCT)
            dY = layer.alloc_dy(B)
            dW = torch.empty(L, K, dtype=torch.bfloat16, device=dev)
            dX = torch.empty(B, d, device=dev)
            loss = torch.zeros(1, device=dev)
            layer.set_profiling(1)
            t = {"fwd": [], "dW": [], "dX": []}
            for it in range(steps + 2):
                flush.fill_(it & 1)
                layer.forward_loss(B, X, idx, W, None, rowptr, col, loss=loss, dY=dY)
                layer.backward(B, X, idx, W, dY, dW=dW, dbias=None, dX=dX)
                torch.cuda.synchronize()
                if it >= 2:
                    t["fwd"].append(layer.kernel_ms(haste.KERNEL_FORWARD)); t["dW"].append(layer.kernel_ms(haste.KERNEL_DW)); t["dX"].append(layer.kernel_ms(haste.KERNEL_DX))
            Wb, ib, dYb, Xb = L * K * 2, NG * K * 4, NG * G * B * 2, B * d * 2
            ab = {"fwd": Wb + ib + Xb + dYb, "dW": dYb + ib + Xb + Wb, "dX": dYb + Wb + ib + B * d * 4}
            out = {"sweep": "config5", "B": B, "G": G, "K": K, "d": d, "L": L, "kernel_family": layer.kernel_family, "flush": "256 MiB fill between iterations"}
            for k in t:
                ms = float(np.median(t[k]))
                out[k] = {"ms": ms, "GB/s": ab[k] / ms / 1e6, "frac_hbm": ab[k] / ms / 1e6 / peaks["hbm"], "TFLOP/s": 2.0 * B * L * K / ms / 1e9,
                          "dense_bottleneck_ms": dense[k], "vs_dense": dense[k] / ms}
            print(json.dumps(out), flush=True)
            del layer, dY, dW, dX, idx
            torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="haste", choices=["haste", "reference"])
    ap.add_argument("--workload", default=WORKLOAD, help="synth.CONFIGS key (default: the 670K-label config the metric is quoted on)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-head", action="store_true", help="time the sparse tail alone")
    ap.add_argument("--two-kernels", action="store_true", help="time the step through haste_forward_loss + haste_backward even where the one-kernel forward + dW exists")
    ap.add_argument("--deterministic", action="store_true", help="create the handles with HASTE_DETERMINISTIC (atomic-free dX)")
    ap.add_argument("--sweep", action="store_true", help="config 5: kernel sweep over B and G at K=64 against the dense bottleneck (one JSON line per point)")
    ap.add_argument("--sweep-B", default="64,256,1024")
    ap.add_argument("--sweep-G", default="1,8,16,32,64,128")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "haste" else args.warmup

    if args.sweep:
        run_sweep(args)
        return
    from paper_2606_01117_b200 import synth
    cfg = synth.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    from paper_2606_01117_b200 import haste     # fails loudly if libhaste.so is missing: no fallback
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    # ---- synthetic inputs of the workload's shape; replicas use their own seed
    inp = synth.make_inputs(cfg, with_head=not args.no_head)
    B, d, L, G, K, Lh = cfg.B, cfg.d, cfg.L_t, cfg.G, cfg.K, cfg.L_h
    use_head = (not args.no_head) and Lh > 0

    tdt = torch.bfloat16 if cfg.dtype == "bf16" else torch.float32
    esz = 2 if cfg.dtype == "bf16" else 4

    def host(key):    # the values both sides consume: bf16 bit patterns (bf16 configs) or the fp32 array (config 1)
        if key in inp.bits:
            return torch.from_numpy(np.ascontiguousarray(inp.bits[key]).view(np.int16)).view(torch.bfloat16)
        return torch.from_numpy(np.ascontiguousarray(getattr(inp, key), dtype=np.float32))

    hX, hrow, hcol = host("X").pin_memory(), torch.from_numpy(inp.rowptr).pin_memory(), torch.from_numpy(inp.col).pin_memory()
    X, rowptr, col = hX.to(dev), hrow.to(dev), hcol.to(dev)
    W, idx = host("W").to(dev), torch.from_numpy(inp.idx).to(dev)
    det = haste.HASTE_DETERMINISTIC if args.deterministic else 0
    layer = haste.HasteLayer(d, L, G, K, B, cfg.dtype, label_offset=Lh, flags=haste.HASTE_IDX_SORTED_DISTINCT | haste.HASTE_XT_FROM_FORWARD | det, device=local)
    layer.validate_index(idx)
    dY = layer.alloc_dy(B)
    dW = torch.empty(L, K, dtype=tdt, device=dev)
    db = torch.empty(L, device=dev)
    dX = torch.empty(B, d, device=dev)
    loss = torch.zeros(2, device=dev)
    if use_head:
        hXh = host("X_head").pin_memory()
        Xh, Wh = hXh.to(dev), host("W_head").to(dev)
        head = haste.HasteHead(d, Lh, B, cfg.dtype, label_offset=0, flags=det, device=local)
        dYh = torch.empty(B, Lh, dtype=tdt, device=dev)
        dWh = torch.empty(Lh, d, dtype=tdt, device=dev)
        dbh = torch.empty(Lh, device=dev)
        dXh = torch.empty(B, d, device=dev)
    launches = [0]

    class Batch:
        """Device buffers of one step's inputs and results.  The device-resident runs use batch 0; the end-to-end run
        alternates between two, so that the copies of one step overlap the kernels of its neighbours."""
        def __init__(self, first):
            self.X, self.rowptr, self.col = (X, rowptr, col) if first else (torch.empty_like(X), torch.empty_like(rowptr), torch.empty_like(col))
            self.dX, self.loss = (dX, loss) if first else (torch.empty_like(dX), torch.zeros_like(loss))
            if use_head:
                self.Xh, self.dXh = (Xh, dXh) if first else (torch.empty_like(Xh), torch.empty_like(dXh))
            self.h_loss, self.h_dX, self.h_dXh = torch.zeros(2).pin_memory(), torch.empty(B, d).pin_memory(), torch.empty(B, d).pin_memory()
            self.ev_in, self.ev_done, self.ev_out = torch.cuda.Event(), torch.cuda.Event(), torch.cuda.Event()

    batches = [Batch(True), Batch(False)]
    s_in, s_out = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)

    # forward + loss + dY + dW + db in ONE kernel where the library has it (bf16, G = 64, B <= 512: tc_fused.cu), then
    # haste_backward for dX only; otherwise haste_forward_loss and haste_backward with all three outputs.  The same results.
    fused_ok = layer.kernel_family == 1 and G == 64 and B <= 512 and not args.two_kernels

    def step(b=batches[0], fused=None):
        n = 0
        if fused_ok if fused is None else fused:
            layer.forward_loss_dw(B, b.X, idx, W, None, b.rowptr, b.col, loss=b.loss[0:1], dY=dY, dW=dW, dbias=db)
            n += layer.last_launch_count
            layer.backward(B, b.X, idx, W, dY, dX=b.dX)
            n += layer.last_launch_count
        else:
            layer.forward_loss(B, b.X, idx, W, None, b.rowptr, b.col, loss=b.loss[0:1], dY=dY)
            n += layer.last_launch_count
            layer.backward(B, b.X, idx, W, dY, dW=dW, dbias=db, dX=b.dX)
            n += layer.last_launch_count
        if use_head:
            head.forward_loss(B, b.Xh, Wh, None, b.rowptr, b.col, loss=b.loss[1:2], dY=dYh)
            n += head.last_launch_count
            head.backward(B, b.Xh, Wh, dYh, dWh=dWh, dbias=dbh, dX=b.dXh)
            n += head.last_launch_count
        launches[0] += n

    e2e_count = [0]

    def step_e2e():
        # one step end to end: inputs from pinned host memory, results back to pinned host memory, through the public
        # calls.  Three streams (copy in, kernels, copy out) and two batches: every step still does all of its copies.
        b = batches[e2e_count[0] & 1]
        e2e_count[0] += 1
        main = torch.cuda.current_stream()
        with torch.cuda.stream(s_in):
            s_in.wait_event(b.ev_done)          # the kernels of the step that last used this batch have read its inputs
            b.X.copy_(hX, non_blocking=True)
            b.rowptr.copy_(hrow, non_blocking=True)
            b.col.copy_(hcol, non_blocking=True)
            if use_head:
                b.Xh.copy_(hXh, non_blocking=True)
            b.ev_in.record(s_in)
        main.wait_event(b.ev_in)
        main.wait_event(b.ev_out)               # the results of that earlier step have left the batch
        step(b)
        b.ev_done.record(main)
        with torch.cuda.stream(s_out):
            s_out.wait_event(b.ev_done)
            b.h_loss.copy_(b.loss, non_blocking=True)
            b.h_dX.copy_(b.dX, non_blocking=True)
            if use_head:
                b.h_dXh.copy_(b.dXh, non_blocking=True)
            b.ev_out.record(s_out)

    def finish_e2e():
        torch.cuda.current_stream().wait_stream(s_out)   # the closing event of the timed region comes after the last copy out

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, finish=None):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            fn()
        if finish is not None:
            finish()
        e1.record()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), dist, dev)

    def rest():
        # every timed pass starts from the same board state: ~50 ms of this load make the board's power management lower the
        # SM clock (see `sustained`), and a pass that follows another directly would start in that state
        torch.cuda.synchronize()
        if args.steps < 20:      # (the few-step runs made under a profiler)
            return
        time.sleep(0.3)
        for _ in range(2):
            step()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    # ---- the timed region of `value`: K steps through the four public calls, nothing else on the stream
    launches[0] = 0
    sampler = ClockSampler(local)
    if rank == 0 and not os.environ.get("HASTE_NO_CLOCKS"):
        sampler.start()
    ms_total = timed(step, args.steps)
    clocks = sampler.stop() if rank == 0 else None
    n_launch = launches[0]
    # ---- a separate pass for the per-kernel breakdown: the library records CUDA events on the launch stream around each
    # kernel (16 records per step, ~2-5 % of the step), so these K steps are not the ones `value` is computed from
    nprof = min(args.steps, 1024)
    rest()
    layer.set_profiling(nprof)
    if use_head:
        head.set_profiling(nprof)
    ms_prof = timed(step, args.steps)
    tail_keys = ("forward_dW", "dX") if fused_ok else ("forward", "dW", "dX")
    kn = {"dX": haste.KERNEL_DX, "prep_fwd": haste.KERNEL_PREP_FWD, "prep_bwd": haste.KERNEL_PREP_BWD, "post_bwd": haste.KERNEL_POST_BWD}
    if fused_ok:
        kn["forward_dW"] = haste.KERNEL_FORWARD          # the one kernel is recorded in the forward slot
    else:
        kn["forward"], kn["dW"] = haste.KERNEL_FORWARD, haste.KERNEL_DW
    kms = {k: [layer.kernel_ms(v, a) for a in range(nprof)] for k, v in kn.items()}
    if use_head:
        kms["head_forward"] = [head.kernel_ms(haste.KERNEL_FORWARD, a) for a in range(nprof)]
        kms["head_backward"] = [head.kernel_ms(haste.KERNEL_DW, a) for a in range(nprof)]
    # ---- forward in logits-only mode: haste_forward_logits, no targets, no loss; the B x L logits are
    # written in the storage dtype (library layout).  Beside it the FLOPs-matched dense bottleneck's forward
    # [B,K] x [L,K]^T in the same dtype through cuBLAS (torch.matmul): a library comparison point, not product code.
    logits_only = None
    if rank == 0 and layer.kernel_family == 1:
        nlog = min(args.steps, nprof, 50)
        for _ in range(2):
            layer.forward_logits(B, X, idx, W, None, dY)
        torch.cuda.synchronize()
        for _ in range(nlog):
            layer.forward_logits(B, X, idx, W, None, dY)
        torch.cuda.synchronize()
        lms = [layer.kernel_ms(haste.KERNEL_FORWARD, a) for a in range(nlog)]
        Lp = (L + 7) // 8 * 8                        # cuBLAS wants 16-byte rows: pad the label count of the comparison
        Hb = torch.randn(B, K, device=dev).to(tdt)
        Wp = torch.zeros(Lp, K, dtype=tdt, device=dev)
        Wp[:L] = W
        Zb = torch.empty(B, Lp, dtype=tdt, device=dev)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nlog)]
        torch.matmul(Hb, Wp.t(), out=Zb)
        for a, b_ in evs:
            a.record(); torch.matmul(Hb, Wp.t(), out=Zb); b_.record()
        torch.cuda.synchronize()
        dms = [a.elapsed_time(b_) for a, b_ in evs]
        lb = L * K * esz + cfg.NG * K * 4 + B * d * esz + cfg.NG * G * B * esz
        logits_only = {"ms": float(np.mean(lms)), "ms_median": float(np.median(lms)), "ms_min": float(np.min(lms)), "alg_bytes": int(lb),
                       "logits_dtype": cfg.dtype, "dense_bottleneck_ms": float(np.median(dms)),
                       "dense_bottleneck_note": "torch.matmul [B,%d] x [L,%d]^T -> [B,L] in %s (cuBLAS), same FLOPs and W/output bytes, no gather" % (K, K, cfg.dtype)}
        del Zb, Hb, Wp
        layer.forward_loss(B, X, idx, W, None, rowptr, col, loss=loss[0:1], dY=dY)     # dY holds dY again for what follows
    # ---- the round-2 calls beside the step (not part of `value`): the SGD-momentum step fused into the dW kernel
    # (haste_backward_sgd, dX skipped here) and the fused top-k forward (haste_forward_topk, k = 5, forward + merge)
    extras = None
    if rank == 0 and layer.kernel_family == 1 and cfg.dtype == "bf16":
        extras = {}
        nx = min(args.steps, nprof, 20)
        try:
            W2, mom = W.clone(), torch.zeros(L, K, device=dev)
            for _ in range(2):
                layer.backward_sgd(B, X, idx, W2, dY, mom, 0.01, 0.9)
            torch.cuda.synchronize()
            for _ in range(nx):
                layer.backward_sgd(B, X, idx, W2, dY, mom, 0.01, 0.9)
            torch.cuda.synchronize()
            t = [layer.kernel_ms(haste.KERNEL_DW, a) for a in range(nx)]
            sb = cfg.NG * G * B * esz + cfg.NG * K * 4 + B * d * esz + 2 * L * K * esz + 2 * L * K * 4
            g = sb / (float(np.mean(t)) * 1e-3) / 1e9
            extras["dW_sgd_fused"] = {"ms": float(np.mean(t)), "ms_median": float(np.median(t)), "ms_min": float(np.min(t)), "alg_bytes": int(sb),
                                      "GB/s": g, "frac_hbm": g / _peaks()["hbm"], "note": "dW never written; W (bf16) and momentum (fp32) read and written in place"}
            del W2, mom
        except haste.HasteError as e:
            extras["dW_sgd_fused"] = {"unsupported": str(e)}
        tv, ti = torch.empty(B, 5, device=dev), torch.empty(B, 5, dtype=torch.int64, device=dev)
        for _ in range(2):
            layer.forward_topk(B, X, idx, W, None, 5, tv, ti)
        torch.cuda.synchronize()
        for _ in range(nx):
            layer.forward_topk(B, X, idx, W, None, 5, tv, ti)
        torch.cuda.synchronize()
        t = [layer.kernel_ms(haste.KERNEL_FORWARD, a) for a in range(nx)]
        extras["forward_topk_k5"] = {"ms": float(np.mean(t)), "ms_median": float(np.median(t)), "ms_min": float(np.min(t)),
                                     "note": "forward kernel with per-thread candidate lists + merge kernel; no [B,L] buffer"}
        # forward + BCE + weight gradient in ONE kernel (haste_forward_loss_dw, first slice) beside the two
        # kernels of the step that it stands for (`kernels.forward` + `kernels.dW`)
        try:
            for _ in range(2):
                layer.forward_loss_dw(B, X, idx, W, None, rowptr, col, loss=loss[0:1], dY=dY, dW=dW, dbias=db)
            torch.cuda.synchronize()
            for _ in range(nx):
                layer.forward_loss_dw(B, X, idx, W, None, rowptr, col, loss=loss[0:1], dY=dY, dW=dW, dbias=db)
            torch.cuda.synchronize()
            t = [layer.kernel_ms(haste.KERNEL_FORWARD, a) for a in range(nx)]
            fb = L * K * esz + cfg.NG * K * 4 + B * d * esz + cfg.NG * G * B * esz + L * K * dW.element_size()
            g = fb / (float(np.mean(t)) * 1e-3) / 1e9
            extras["forward_dw_fused"] = {"ms": float(np.mean(t)), "ms_median": float(np.median(t)), "ms_min": float(np.min(t)), "alg_bytes": int(fb),
                                          "GB/s": g, "frac_hbm": g / _peaks()["hbm"], "launches": int(layer.last_launch_count),
                                          "note": "one kernel for forward + loss + dY + dW + db where it exists (G = 64, B <= 512), else the two kernels; dY written once, never read back"}
        except haste.HasteError as e:
            extras["forward_dw_fused"] = {"unsupported": str(e)}
        # ... and the two kernels that call stands for, timed the same way (haste_forward_loss, haste_backward for dW and db)
        for _ in range(2):
            layer.forward_loss(B, X, idx, W, None, rowptr, col, loss=loss[0:1], dY=dY)
            layer.backward(B, X, idx, W, dY, dW=dW, dbias=db)
        torch.cuda.synchronize()
        for _ in range(nx):
            layer.forward_loss(B, X, idx, W, None, rowptr, col, loss=loss[0:1], dY=dY)
            layer.backward(B, X, idx, W, dY, dW=dW, dbias=db)
        torch.cuda.synchronize()
        tf_ = [layer.kernel_ms(haste.KERNEL_FORWARD, a) for a in range(nx)]
        tw_ = [layer.kernel_ms(haste.KERNEL_DW, a) for a in range(nx)]
        ab2 = _alg_bytes(cfg, dw_bytes=dW.element_size())
        extras["forward_then_dW"] = {"forward_ms": float(np.mean(tf_)), "dW_ms": float(np.mean(tw_)), "ms": float(np.mean(tf_) + np.mean(tw_)),
                                     "forward_frac_hbm": ab2["forward"] / (float(np.mean(tf_)) * 1e-3) / 1e9 / _peaks()["hbm"],
                                     "dW_frac_hbm": ab2["dW"] / (float(np.mean(tw_)) * 1e-3) / 1e9 / _peaks()["hbm"],
                                     "note": "the forward kernel and the dW kernel on their own, alternating"}
    layer.set_profiling(0)
    if use_head:
        head.set_profiling(0)
    for _ in range(2):
        step_e2e()
    rest()
    ms_e2e = timed(step_e2e, args.steps, finish_e2e)
    # the pipelined run must have brought back the results of the device-resident run (same inputs every step)
    for b in batches:
        if not torch.equal(b.h_loss, loss.cpu()) or not torch.allclose(b.h_dX, dX.cpu(), rtol=1e-3, atol=1e-6):
            raise RuntimeError("bench.py: the end-to-end run returned different results from the device-resident run")

    # ---- sustained operation, reported beside `value`: after ~50 ms of this load the board's power management lowers the SM
    # clock (sw_power_cap is reported at ~330 W), so a long region is slower per step than the default K = 50 one
    sustained = None
    if 20 <= args.steps < 200:      # (not in the few-step runs made under a profiler)
        s2 = ClockSampler(local)
        if rank == 0 and not os.environ.get("HASTE_NO_CLOCKS"):
            s2.start()
        ms_sus = timed(step, 200)
        c2 = s2.stop() if rank == 0 else None
        sustained = {"steps": 200, "ms_per_step": ms_sus / 200, "clocks": c2,
                     "note": "200 more steps timed the same way after everything else; not the region `value` is computed from"}
    # ---- the same step through the two separate kernels (haste_forward_loss, then haste_backward with dW, db and dX), where the
    # timed step used the one-kernel route: the same outputs, 0.7 GB more HBM traffic per step.  Reported beside `value`.
    two_kernel_step = None
    if 20 <= args.steps < 200 and fused_ok:
        def step_2(b=batches[0]):
            step(b, fused=False)
        rest()
        for _ in range(3):
            step_2()
        torch.cuda.synchronize()
        time.sleep(0.3)
        ms_2 = timed(step_2, args.steps)
        ms_2s = timed(step_2, 200)
        two_kernel_step = {"ms_per_step": ms_2 / args.steps, "steps": args.steps, "sustained_ms_per_step": ms_2s / 200, "sustained_steps": 200,
                           "note": "the step through haste_forward_loss + haste_backward(dW, db, dX); timed like `value` and like `sustained`"}
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peaks = _peaks()
    tail_f, head_f = _flops(cfg)
    step_flops = 3 * tail_f + (3 * head_f if use_head else 0)
    ms_step = ms_total / args.steps
    value = whole_job_tflops(world, step_flops, ms_step)
    e2e_value = whole_job_tflops(world, step_flops, ms_e2e / args.steps)
    ab = _alg_bytes(cfg)
    SPEC_HBM, SPEC_BF16 = 8000.0, 2250.0          # B200 nominal: HBM3e GB/s, dense bf16 TFLOP/s
    kernels = {}
    for k in tail_keys:
        mean, med = float(np.mean(kms[k])), float(np.median(kms[k]))
        gbs = ab[k] / (mean * 1e-3) / 1e9
        kernels[k] = {"ms": mean, "ms_median": med, "ms_min": float(np.min(kms[k])), "GB/s": gbs, "frac_hbm": gbs / peaks["hbm"],
                      "frac_hbm_spec": gbs / SPEC_HBM, "TFLOP/s": (2 if k == "forward_dW" else 1) * tail_f / (mean * 1e-3) / 1e12, "alg_bytes": ab[k]}
    for k in kms:
        if k not in kernels:
            kernels[k] = {"ms": float(np.mean(kms[k])), "ms_median": float(np.median(kms[k])), "ms_min": float(np.min(kms[k]))}
    if use_head:
        for k, fl in (("head_forward", head_f), ("head_backward", 2 * head_f)):
            tf = fl / (kernels[k]["ms"] * 1e-3) / 1e12
            kernels[k].update({"TFLOP/s": tf, "frac_tensor": tf / peaks["bf16_sustained"], "frac_tensor_burst": tf / peaks["bf16"],
                               "frac_tensor_spec": tf / SPEC_BF16})
    if logits_only is not None:
        g = logits_only["alg_bytes"] / (logits_only["ms"] * 1e-3) / 1e9
        logits_only.update({"GB/s": g, "frac_hbm": g / peaks["hbm"], "frac_hbm_spec": g / SPEC_HBM})
        kernels["forward_logits_only"] = logits_only
    dom = max(tail_keys, key=lambda k: kernels[k]["ms"])
    # DRAM bytes per launch of that kernel from the committed `ncu --set full` capture of this round.  The record names the
    # kernel and carries the SHA-256 of the kernel source it was captured from: a stale record (source changed since) gives null.
    traffic, traffic_src = None, None
    try:
        import hashlib
        tj = json.load(open(os.path.join(ROOT, "profiles", "r02_ncu_traffic.txt")))
        rec = tj.get(dom) if tj.get("workload") == args.workload else None
        if rec:
            h = hashlib.sha256(open(os.path.join(ROOT, rec["source"]), "rb").read()).hexdigest()
            if h == rec["source_sha256"]:
                traffic, traffic_src = rec["dram_bytes"], {"kernel": rec["kernel"], "capture": rec["capture"], "source": rec["source"]}
    except Exception:
        traffic = None
    roofline = {"kernel": dom, "bound": "hbm", "achieved": kernels[dom]["GB/s"], "peak": peaks["hbm"], "unit": "GB/s",
                "frac": kernels[dom]["GB/s"] / peaks["hbm"], "frac_spec": kernels[dom]["GB/s"] / SPEC_HBM, "peak_spec": SPEC_HBM,
                "traffic": traffic, "traffic_unit": "bytes per launch (ncu dram read+write)", "traffic_from": traffic_src,
                "algorithmic_bytes": ab[dom], "peak_source": peaks["source"] + " (burst copy)",
                "share_of_step": kernels[dom]["ms"] / (ms_prof / args.steps),
                "timing": "CUDA events on the launch stream around the kernel, mean over the K steps of a separate profiled pass"}
    pass_mb = (L * K * esz >> 20, cfg.NG * G * B * esz >> 20)
    if sum(pass_mb) > 126:
        l2_note = "inputs larger than L2 (per pass W %d MB + dY %d MB vs 126 MB L2); no explicit flush" % pass_mb
    else:
        l2_note = "inputs SMALLER than L2 (per pass W %d MB + dY %d MB vs 126 MB L2) and no flush: an L2-resident parity-size config, not a roofline measurement" % pass_mb
    h2d = hX.numel() * esz + hrow.numel() * 4 + hcol.numel() * 4 + (hXh.numel() * esz if use_head else 0)
    d2h = 8 + B * d * 4 * (2 if use_head else 1)
    out = {
        "metric": "sparse_layer_fwd_bwd_tflops_670k", "value": value, "unit": "TFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": cfg.dtype, "data": "synthetic",
        "config": {"workload": "config3_670k" if args.workload == "670k" else args.workload, "B": B, "d": d, "L_tail": L, "L_head": Lh if use_head else 0,
                   "G": G, "K": K, "replicas": world, "l2": l2_note,
                   "step_route": ("haste_forward_loss_dw (forward + loss + dY + dW + db in one kernel) + haste_backward (dX)" if fused_ok
                                  else "haste_forward_loss + haste_backward (dW, db, dX)") + (" + head forward + head backward" if use_head else ""),
                   "kernel_family": {"tail": layer.kernel_family, "head": head.kernel_family if use_head else None}, "deterministic": bool(args.deterministic)},
        "e2e": {"value": e2e_value, "unit": "TFLOP/s", "ms_per_step": ms_e2e / args.steps, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "note": "copies on their own streams, two sets of device buffers; no per-kernel events"},
        "gpu_launches": int(n_launch), "clocks": clocks, "roofline": roofline, "kernels": kernels,
        "profiled_pass": {"ms_per_step": ms_prof / args.steps,
                          "note": "the same K steps repeated with the library's per-kernel CUDA events on; `kernels` and `roofline` come from this pass, `value` does not"},
        "loss": [float(v) for v in loss.cpu().tolist()],
    }
    if extras:
        out["extras"] = extras
    if sustained:
        sustained["value"] = whole_job_tflops(world, step_flops, sustained["ms_per_step"])
        out["sustained"] = sustained
    if two_kernel_step:
        two_kernel_step["value"] = whole_job_tflops(world, step_flops, two_kernel_step["ms_per_step"])
        two_kernel_step["sustained_value"] = whole_job_tflops(world, step_flops, two_kernel_step["sustained_ms_per_step"])
        out["step_two_kernels"] = two_kernel_step
    if not args.no_cpu_baseline and world == 1:
        out["cpu_baseline"] = cpu_baseline(cfg)
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
