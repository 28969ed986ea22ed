#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path over one synthetic clip:
for every sliding window, `layers` alternating frame/global attention layers (mf_window_attention),
then mf_chain_poses over all windows, then mf_motion_focus (focus map + guided depth) for every frame.

Default workload: BASELINE.json configs[3] (campus-shaped, W=32 stride 16, 1800 frames at 1920x1080,
S=24864 tokens/window, 24 layers, H=16, D=64, bf16) -- the config the metric "frames/sec at W=32" is
quoted on.  Prints ONE JSON line.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

L2_BYTES = 126 * 2 ** 20


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="index into BASELINE.json configs (default 3 = campus, W=32); 5..11 = the rows of the paper's Table 2 (synth.CONFIGS)")
    ap.add_argument("--windows-per-launch", type=int, default=4)
    ap.add_argument("--focus-chunk", type=int, default=300, help="frames per mf_motion_focus call")
    ap.add_argument("--max-windows", type=int, default=0, help="debug: truncate the clip to this many windows")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-stream", action="store_true", help="skip the per-window streaming latency measurement (SURVEY 8(f) NEXT-2)")
    ap.add_argument("--no-d128", action="store_true", help="skip the head_dim 128 attention measurement (SURVEY 8(f) NEXT-3)")
    ap.add_argument("--no-block", action="store_true", help="skip the whole-transformer-block measurement (SURVEY 8(f) NEXT-1)")
    ap.add_argument("--no-per-config", action="store_true", help="skip the short runs of the other BASELINE.json configs (SURVEY 8(d))")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return dict(hbm=d["hbm_gbs"], tf_burst=d["bf16_tflops"], tf_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    source="measured")
    return dict(hbm=6650.0, tf_burst=1590.0, tf_sustained=1400.0, source="fallback")


TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_ncu_attn_traffic.csv")


def ncu_traffic(cfg_idx, windows_per_launch):
    """DRAM bytes per GLOBAL attention launch (dram__bytes_read.sum + dram__bytes_write.sum) of the committed `ncu --set full`
    capture of this launch shape, read from profiles/r2_ncu_attn_traffic.csv (text; written from the .ncu-rep, see the .md
    beside it).  It is NOT measured in this run (ncu cannot run inside the timed bench); no capture of the shape -> None."""
    try:
        with open(TRAFFIC_CSV) as f:
            for ln in f:
                parts = [x.strip() for x in ln.split(",")]
                if len(parts) >= 4 and parts[0].isdigit() and (int(parts[0]), int(parts[1])) == (cfg_idx, windows_per_launch):
                    return float(parts[2]) + float(parts[3])
    except OSError:
        pass
    return None


class ClockSampler:
    """Polls nvidia-smi during the timed region (B200_PROFILING.md clocks line)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True).start()
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            try:
                pw.append(float(parts[2]))
            except ValueError:
                pass
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        busy = [x for x in sm if x > 0.5 * (mx[0] if mx else 1)] or sm
        return {"sm_mhz": busy[len(busy) // 2] if busy else None, "sm_max_mhz": mx[0] if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "power_w_max": max(pw) if pw else None}


class Workload:
    def __init__(self, cfg_idx, args, device):
        import torch
        from paper_2601_07154_b200 import api, synth
        self.torch, self.api, self.synth = torch, api, synth
        cfg = dict(synth.CONFIGS[cfg_idx])
        self.cfg, self.cfg_idx, self.device = cfg, cfg_idx, device
        self.W, self.P, self.H, self.D = cfg["W"], cfg["P"], cfg["H"], cfg["D"]
        self.S = self.W * self.P
        self.stride, self.layers = cfg["stride"], cfg["layers"]
        self.N = cfg["N"]
        self.Nw = api.num_windows(self.N, self.W, self.stride)
        if args.max_windows and args.max_windows < self.Nw:
            self.Nw = args.max_windows
            self.N = (self.Nw - 1) * self.stride + self.W
        self.B = max(1, min(args.windows_per_launch, self.Nw))
        self.chunk = max(1, min(args.focus_chunk, self.N))
        self.width, self.height = cfg["width"], cfg["height"]
        self.n_points = 15
        # algorithmic work
        self.flops_global = 4.0 * self.S * self.S * self.H * self.D                  # per window-layer
        self.flops_frame = 4.0 * self.W * self.P * self.P * self.H * self.D
        self.n_global = self.layers // 2 if self.layers > 1 else 1      # tiny config: its one layer is GLOBAL (BJ configs[0])
        self.n_frame = self.layers - self.n_global
        self.flops_step = self.Nw * (self.n_global * self.flops_global + self.n_frame * self.flops_frame)
        self.focus_bytes_step = 12.0 * self.N * self.width * self.height

    @staticmethod
    def launches_per_step(cfg_idx, args, api):
        """Kernels of ours launched by one step_device() pass: one per (launch batch, layer), the pose chain, and 3 per focus call
        (tables, norm, render); a GLOBAL layer of a long sequence is two kernels (attention_kernels)."""
        w = Workload.__new__(Workload)
        Workload.__init__(w, cfg_idx, args, None)
        batches = (w.Nw + w.B - 1) // w.B
        return batches * (w.n_global * Workload.attention_kernels(w.S, w.D) + w.n_frame * Workload.attention_kernels(w.P, w.D)) \
            + 1 + 3 * ((w.N + w.chunk - 1) // w.chunk)

    @staticmethod
    def attention_kernels(seq_len, head_dim):
        """Kernels of one mf_window_attention call: head_dim 64 sequences of 32 KV tiles and more run the key-norm pass of the
        score bound (key_norm_max_kernel), window_attention_split_kernel (the CTAs within the bound) and window_attention_kernel
        (the others; csrc/attention.cu, attention_split.cu)."""
        return 3 if head_dim == 64 and (seq_len + 127) // 128 >= 32 else 1

    @staticmethod
    def flops_per_step(cfg_idx, args, api):
        w = Workload.__new__(Workload)
        Workload.__init__(w, cfg_idx, args, None)
        return w.flops_step

    def release_host(self):
        for name in ("hq", "hk", "hv", "ho", "hlocal", "hdepth", "hout", "hstreams"):
            if hasattr(self, name):
                delattr(self, name)

    # ---- device-resident inputs ----
    def setup_device(self):
        torch, synth = self.torch, self.synth
        dev = self.device
        self.q, self.k, self.v = synth.qkv(self.Nw, self.S, self.H, self.D, synth.seed_for(self.cfg_idx, 0), device=dev)
        self.o = [torch.empty((self.B, self.S, self.H, self.D), device=dev, dtype=torch.bfloat16) for _ in range(2)]
        traj = synth.trajectory(self.cfg, synth.seed_for(self.cfg_idx, 1), self.N)
        self.local_np = synth.local_windows(traj, self.W, self.api.window_starts(self.N, self.W, self.stride), seed=synth.seed_for(self.cfg_idx, 2),
                                            perturb_rot=1e-3, perturb_t=1e-3)
        self.local = torch.from_numpy(self.local_np).to(dev)
        self.depth = synth.depth(self.N, self.height, self.width, synth.seed_for(self.cfg_idx, 3), device=dev)
        self.fmap = torch.empty_like(self.depth)
        self.guided = torch.empty_like(self.depth)
        self.params = self.api.focus_params(n_points=self.n_points, sigma=self.cfg["sigma"])
        need = self.api.lib().mf_motion_focus_workspace_size(self.chunk, self.width, self.height, self.n_points)
        self.ws = torch.empty((need,), device=dev, dtype=torch.uint8)
        self.launches = 0

    def step_device(self, ev_global=None, ev_focus=None):
        """One full pass, everything resident in HBM.  ev_* collect (start, end) CUDA event pairs."""
        torch, api = self.torch, self.api
        launches = 0
        for b0 in range(0, self.Nw, self.B):
            b1 = min(b0 + self.B, self.Nw)
            qb, kb, vb = self.q[b0:b1], self.k[b0:b1], self.v[b0:b1]
            for layer in range(self.layers):
                mode = api.ATTN_FRAME if (layer % 2 == 0 and self.layers > 1) else api.ATTN_GLOBAL   # reading A3
                out = self.o[layer % 2][: b1 - b0]
                if ev_global is not None and mode == api.ATTN_GLOBAL:
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    api.window_attention(qb, kb, vb, self.W, self.P, mode, out=out)
                    e1.record()
                    ev_global.append((e0, e1, b1 - b0))
                else:
                    api.window_attention(qb, kb, vb, self.W, self.P, mode, out=out)
                launches += 1
        poses = api.chain_poses(self.local, self.stride, self.N)
        launches += 1
        c = self.cfg
        for f0 in range(0, self.N, self.chunk):
            f1 = min(f0 + self.chunk, self.N)
            if ev_focus is not None:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
            api.motion_focus(poses, c["fx"], c["fy"], c["cx"], c["cy"], self.width, self.height, self.params,
                             depth=self.depth[f0:f1], render_begin=f0, render_end=f1, workspace=self.ws,
                             out={"focus_map": self.fmap[f0:f1], "guided_depth": self.guided[f0:f1]})
            if ev_focus is not None:
                e1.record()
                ev_focus.append((e0, e1, f1 - f0))
            launches += 3
        self.launches = launches
        return poses

    # ---- end-to-end through the host-buffer C ABI ----
    def setup_host(self):
        """Pinned host buffers for the end-to-end path.  The blocking *_host entry points are called from four host
        threads (two for the window batches, two for the focus chunks), each on its own CUDA stream, so one call's
        PCIe copies overlap another call's kernels; every byte of every window / frame still crosses PCIe once."""
        torch = self.torch
        pin = lambda t: t.cpu().pin_memory()
        self.hq, self.hk, self.hv = pin(self.q[: self.B]), pin(self.k[: self.B]), pin(self.v[: self.B])
        self.ho = [torch.empty_like(self.hq).pin_memory() for _ in range(2)]
        self.hlocal = torch.from_numpy(self.local_np).pin_memory()
        self.hchunk = max(1, min(self.chunk, 100))
        self.hdepth = pin(self.depth[: self.hchunk])
        self.hout = [{"focus_map": torch.empty_like(self.hdepth).pin_memory(),
                      "guided_depth": torch.empty_like(self.hdepth).pin_memory(),
                      "global_w2c": torch.empty((self.N, 4, 4), dtype=torch.float64).pin_memory()} for _ in range(2)]
        self.hstreams = [torch.cuda.Stream(device=self.device) for _ in range(4)]
        tok = self.S * self.H * self.D * 2
        img = self.width * self.height * 4
        n_chunks = (self.N + self.hchunk - 1) // self.hchunk
        self.h2d = self.Nw * 3 * tok + self.N * img + n_chunks * self.hlocal.numel() * 4
        self.d2h = self.Nw * tok + 2 * self.N * img + n_chunks * self.N * 128 + self.N * 12

    def step_host(self):
        from concurrent.futures import ThreadPoolExecutor
        api, c, torch = self.api, self.cfg, self.torch
        batches = list(range(0, self.Nw, self.B))
        chunks = list(range(0, self.N, self.hchunk))

        def attn_worker(wid):
            torch.cuda.set_device(self.device)
            with torch.cuda.stream(self.hstreams[wid]):
                for b0 in batches[wid::2]:
                    nb = min(self.B, self.Nw - b0)
                    api.window_attention_host(self.hq[:nb], self.hk[:nb], self.hv[:nb], self.W, self.P,
                                              api.ATTN_FRAME if self.layers > 1 else api.ATTN_GLOBAL,
                                              out=self.ho[wid][:nb], num_layers=self.layers)

        def focus_worker(wid):
            torch.cuda.set_device(self.device)
            with torch.cuda.stream(self.hstreams[2 + wid]):
                for f0 in chunks[wid::2]:
                    f1 = min(f0 + self.hchunk, self.N)
                    n = f1 - f0
                    o = self.hout[wid]
                    api.chain_and_focus_host(self.hlocal, self.stride, self.N, c["fx"], c["fy"], c["cx"], c["cy"], self.width,
                                             self.height, self.params, depth=self.hdepth[:n], render_begin=f0, render_end=f1,
                                             out={"focus_map": o["focus_map"][:n], "guided_depth": o["guided_depth"][:n],
                                                  "global_w2c": o["global_w2c"]})

        with ThreadPoolExecutor(4) as ex:
            futs = [ex.submit(attn_worker, 0), ex.submit(attn_worker, 1), ex.submit(focus_worker, 0), ex.submit(focus_worker, 1)]
            for f in futs:
                f.result()


def measure_block(wl, torch, api):
    """SURVEY 8(f) NEXT-1 (not part of the headline step): one FRAME + one GLOBAL pre-norm transformer block
    (mf_block_forward: LN, QKV GEMM, window attention, out-proj GEMM + residual, LN, fc1 GEMM + GELU, fc2 GEMM + residual)
    on one launch batch of windows, d = H*D, hidden = 4d, seeded synthetic weights."""
    from paper_2601_07154_b200 import synth
    d, dh = wl.H * wl.D, 4 * wl.H * wl.D
    tokens = wl.B * wl.S
    x = synth.tokens(tokens, d, synth.seed_for(wl.cfg_idx, 6), device=wl.device)
    wts = synth.block_weights(d, dh, synth.seed_for(wl.cfg_idx, 7), device=wl.device)
    need = api.lib().mf_block_workspace_size(wl.B, wl.W, wl.P, d, dh)
    ws = torch.empty((need,), device=wl.device, dtype=torch.uint8)
    y = torch.empty_like(x)
    gemm_flops = 2.0 * tokens * (3 * d * d + d * d + 2 * d * dh)
    out = {"what": "mf_block_forward on one launch batch (SURVEY 8(f) NEXT-1; not in the headline step)",
           "tokens": tokens, "d_model": d, "d_hidden": dh, "gemm_flops_per_block": gemm_flops}
    for name, mode, aflops in (("frame", api.ATTN_FRAME, wl.flops_frame), ("global", api.ATTN_GLOBAL, wl.flops_global)):
        for _ in range(2):
            api.block_forward(x, wts, wl.B, wl.W, wl.P, wl.H, mode, out=y, workspace=ws)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(3):
            api.block_forward(x, wts, wl.B, wl.W, wl.P, wl.H, mode, out=y, workspace=ws)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 3
        out[name + "_block_ms"] = ms
        out[name + "_block_tflops"] = (gemm_flops + aflops * wl.B) / (ms * 1e-3) / 1e12
    pair_ms = out["frame_block_ms"] + out["global_block_ms"]
    out["frames_per_s_full_blocks"] = wl.N / (pair_ms * 1e-3 * (wl.layers // 2) * ((wl.Nw + wl.B - 1) // wl.B))
    return out


def measure_d128(wl, torch, api, peak_sustained):
    """SURVEY 8(f) NEXT-3 (not part of the headline step): the GLOBAL attention launch of this workload at head_dim 128 with
    half the heads (same d_model, same S, same windows per launch), 0.5 s of back-to-back launches after warm-up."""
    from paper_2601_07154_b200 import synth
    heads = max(1, wl.H * wl.D // 128)
    q, k, v = synth.qkv(wl.B, wl.S, heads, 128, synth.seed_for(wl.cfg_idx, 8), device=wl.device)
    o = torch.empty_like(q)
    flops = 4.0 * wl.S * wl.S * heads * 128 * wl.B
    for _ in range(3):
        api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_GLOBAL, out=o)
    torch.cuda.synchronize()
    n = 50 if wl.S >= 8192 else 200
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n):
        api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_GLOBAL, out=o)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / n
    tf = flops / (ms * 1e-3) / 1e12
    return {"what": "mf_window_attention GLOBAL at head_dim 128 (SURVEY 8(f) NEXT-3; not in the headline step)", "heads": heads,
            "seq_len": wl.S, "windows_per_launch": wl.B, "launches": n, "ms_per_launch": ms, "tflops": tf,
            "frac_of_sustained_peak": tf / peak_sustained}


def measure_exact_path(wl, torch, api, peak_sustained):
    """The GLOBAL launch of this workload on PEAKED inputs (queries x 8: every row's score bound is above the 32 log2 units of
    csrc/attention.cu, so every CTA is flagged and runs window_attention_kernel's exact online softmax): the rate a caller gets whose
    logits are not bounded like the bench's N(0,1) / qk-normalised tokens are.  Not part of the headline step."""
    from paper_2601_07154_b200 import synth
    q, k, v = synth.qkv(wl.B, wl.S, wl.H, wl.D, synth.seed_for(wl.cfg_idx, 11), device=wl.device)
    q = (q.float() * 8.0).to(torch.bfloat16)
    o = torch.empty_like(q)
    flops = wl.flops_global * wl.B
    for _ in range(3):
        api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_GLOBAL, out=o)
    torch.cuda.synchronize()
    n = 30 if wl.S >= 8192 else 200
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n):
        api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_GLOBAL, out=o)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / n
    tf = flops / (ms * 1e-3) / 1e12
    return {"what": "mf_window_attention GLOBAL on queries x 8 (score bound exceeded everywhere: exact online-softmax path; not in the "
                    "headline step)", "windows_per_launch": wl.B, "launches": n, "ms_per_launch": ms, "tflops": tf,
            "frac_of_sustained_peak": tf / peak_sustained}


def measure_one_wave(wl, torch, api, peak_sustained):
    """the tiny config is launch-bound at one window, so its GLOBAL layer is also timed with 148 windows per launch
    (one window-head per SM and q-block wave)."""
    from paper_2601_07154_b200 import synth
    nw = 148
    q, k, v = synth.qkv(nw, wl.S, wl.H, wl.D, synth.seed_for(wl.cfg_idx, 10), device=wl.device)
    o = torch.empty_like(q)
    for _ in range(3):
        api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_GLOBAL, out=o)
    torch.cuda.synchronize()
    n = 100
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n):
        api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_GLOBAL, out=o)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / n
    tf = wl.flops_global * nw / (ms * 1e-3) / 1e12
    return {"what": "GLOBAL layer of this config with 148 windows per launch (SURVEY 8(d))", "windows_per_launch": nw,
            "us_per_launch": ms * 1e3, "tflops": tf, "frac_of_sustained_peak": tf / peak_sustained}


def measure_streaming(wl, torch, api):
    """SURVEY 8(f) NEXT-2 (not part of the headline step): the path one window at a time, as a stream would see it.
    Per window: its q,k,v into static buffers, 24 attention launches, mf_chain_poses_step, the new poses appended to a
    rolling pose buffer, mf_motion_focus for the `stride` new frames.  Timed eagerly and as one replayed CUDA graph."""
    from paper_2601_07154_b200 import synth
    c, dev = wl.cfg, wl.device
    synth_seed = synth.seed_for(wl.cfg_idx, 9)
    m = wl.stride
    ring_len = wl.W + 32
    q, k, v = (torch.empty_like(t[:1]) for t in (wl.q, wl.k, wl.v))
    o = [torch.empty_like(q) for _ in range(2)]
    win = torch.empty((wl.W, 4, 4), device=dev, dtype=torch.float32)
    state = api.chain_state(dev)
    ring = torch.zeros((ring_len, 4, 4), device=dev, dtype=torch.float64)
    new = torch.empty((m, 4, 4), device=dev, dtype=torch.float64)
    depth = wl.depth[:m]
    fmap, guided = torch.empty_like(depth), torch.empty_like(depth)
    ws = torch.empty((api.lib().mf_motion_focus_workspace_size(m, wl.width, wl.height, wl.n_points),), device=dev, dtype=torch.uint8)

    def load(n):
        q.copy_(wl.q[n:n + 1]); k.copy_(wl.k[n:n + 1]); v.copy_(wl.v[n:n + 1]); win.copy_(wl.local[n])

    def attention():
        for layer in range(wl.layers):
            api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_FRAME if layer % 2 == 0 else api.ATTN_GLOBAL, out=o[layer % 2])

    def step(first=False, with_attention=True):
        if with_attention:
            attention()
        if first:
            full = api.chain_poses_step(win, state, first=True)
            ring[-wl.W:].copy_(full)
            return
        api.chain_poses_step(win, state, new_frames=m, out=new)
        ring.copy_(torch.cat([ring[m:], new]))
        api.motion_focus(ring, c["fx"], c["fy"], c["cx"], c["cy"], wl.width, wl.height, wl.params, depth=depth,
                         render_begin=ring_len - m, render_end=ring_len, workspace=ws,
                         out={"focus_map": fmap, "guided_depth": guided})

    def timed(fn, windows):
        ts = []
        for n in windows:
            load(n)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        ts.sort()
        return ts[len(ts) // 2]

    load(0); step(first=True)
    load(1); step()
    torch.cuda.synchronize()
    eager_ms = timed(step, range(2, 5))
    graph = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream(device=dev)
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()                                               # warm-up on the capture stream
        torch.cuda.synchronize()
        with torch.cuda.graph(graph, stream=side):
            step()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    graph_ms = timed(graph.replay, range(5, 8))

    # Overlapped form: the attention stack of window n+1 runs on the main stream while the chain step and the focus render of
    # window n run on a second stream (two graphs; q,k,v are only touched on the main stream, the window-local poses only on
    # the second one).  Steady-state time per window over 6 windows back to back, against the single graph timed the same way.
    main = torch.cuda.current_stream()
    tail_stream = torch.cuda.Stream(device=dev)
    g_attn, g_tail = torch.cuda.CUDAGraph(), torch.cuda.CUDAGraph()
    side.wait_stream(main)
    with torch.cuda.stream(side):
        with torch.cuda.graph(g_attn, stream=side):
            attention()
        with torch.cuda.graph(g_tail, stream=side):
            step(with_attention=False)
    main.wait_stream(side)
    torch.cuda.synchronize()

    def run_serial(n):
        load(n)
        graph.replay()

    def run_overlapped(n):
        q.copy_(wl.q[n:n + 1]); k.copy_(wl.k[n:n + 1]); v.copy_(wl.v[n:n + 1])
        g_attn.replay()
        done = torch.cuda.Event()
        done.record(main)
        with torch.cuda.stream(tail_stream):
            tail_stream.wait_event(done)
            win.copy_(wl.local[n])
            g_tail.replay()

    def back_to_back(fn, windows):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(main)
        for n in windows:
            fn(n)
        main.wait_stream(tail_stream)
        e1.record(main)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / len(windows)

    # The same window step with the depth stream of Fig. 3: the window's model-resolution depth (518x294) is scale-aligned on the
    # overlap (mf_align_depth_step), the new frames are emitted and the render interpolates them (mf_motion_focus_upsampled).
    gd = torch.Generator(device=dev).manual_seed(synth_seed)
    dwin = [torch.rand((wl.W, 294, 518), generator=gd, device=dev) * 29.0 + 1.0 for _ in range(2)]
    dstate = api.align_depth_state(dev)
    dnew = torch.empty((m, 294, 518), device=dev, dtype=torch.float32)
    api.align_depth_step(dwin[0], dstate, first=True)

    def step_depth():
        attention()
        api.chain_poses_step(win, state, new_frames=m, out=new)
        ring.copy_(torch.cat([ring[m:], new]))
        api.align_depth_step(dwin[1], dstate, prev_window=dwin[0], new_frames=m, out=dnew)
        api.motion_focus_upsampled(ring, c["fx"], c["fy"], c["cx"], c["cy"], wl.width, wl.height, dnew, wl.params,
                                   render_begin=ring_len - m, render_end=ring_len, workspace=ws,
                                   out={"focus_map": fmap, "guided_depth": guided})

    g_depth = torch.cuda.CUDAGraph()
    side.wait_stream(main)
    with torch.cuda.stream(side):
        step_depth()
        torch.cuda.synchronize()
        with torch.cuda.graph(g_depth, stream=side):
            step_depth()
    main.wait_stream(side)
    torch.cuda.synchronize()
    depth_graph_ms = timed(g_depth.replay, range(5, 8))

    nwin = list(range(2, min(wl.Nw, 8)))
    back_to_back(run_overlapped, nwin[:2])
    serial_ms = back_to_back(run_serial, nwin)
    overlap_ms = back_to_back(run_overlapped, nwin)
    return {"what": f"one window at a time (SURVEY 8(f) NEXT-2; not in the headline step): {wl.layers} attention launches + "
                    "mf_chain_poses_step + rolling pose buffer + mf_motion_focus of the new frames",
            "new_frames_per_window": m, "eager_ms_per_window": eager_ms, "graph_ms_per_window": graph_ms,
            "graph_back_to_back_ms_per_window": serial_ms, "two_stream_overlap_ms_per_window": overlap_ms,
            "graph_ms_per_window_with_depth_alignment_and_upsampling": depth_graph_ms,
            "frames_per_s_streaming": m / (graph_ms * 1e-3),
            "kernels_per_window": wl.n_global * Workload.attention_kernels(wl.S, wl.D) + wl.n_frame * Workload.attention_kernels(wl.P, wl.D) + 1 + 3}


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample(cfg_idx, wl_dims, rows=4096):
    """Times the oracle, as it stands, on a bounded sample of the same workload (host cores) and
    extrapolates to the whole clip.  Returns (frames_per_s, seconds_of_sample, description, cores)."""
    import numpy as np
    import torch
    from threadpoolctl import threadpool_info
    from oracle import attention as oa
    from oracle import chain as oc
    from oracle import points as op
    from oracle import render as orr
    from oracle import windows as ow
    from paper_2601_07154_b200 import synth
    cfg = synth.CONFIGS[cfg_idx]
    W, P, H, D, S, Nw, N, layers = (wl_dims[k] for k in ("W", "P", "H", "D", "S", "Nw", "N", "layers"))
    q, k, v = (t.float().numpy().astype(np.float64) for t in synth.qkv(1, S, H, D, synth.seed_for(cfg_idx, 0)))
    rows = min(rows, S)
    sel = np.sort(np.random.default_rng(0).choice(S, rows, replace=False))
    t0 = time.perf_counter()
    oa.window_attention(q, k, v, W, P, oa.GLOBAL, rows=sel)
    t_global = time.perf_counter() - t0
    t0 = time.perf_counter()
    oa.window_attention(q, k, v, W, P, oa.FRAME, rows=np.arange(P))
    t_frame = time.perf_counter() - t0
    traj = synth.trajectory(cfg, synth.seed_for(cfg_idx, 1), N)
    loc = synth.local_windows(traj, W, ow.window_starts(N, W, cfg["stride"]), seed=synth.seed_for(cfg_idx, 2), perturb_rot=1e-3, perturb_t=1e-3)
    t0 = time.perf_counter()
    poses = oc.chain_poses(loc.tolist(), W, cfg["stride"], N)
    frames = op.motion_points(poses, cfg["fx"], cfg["fy"], cfg["cx"], cfg["cy"], cfg["width"], cfg["height"], 15, cfg["sigma"])
    t_pose = time.perf_counter() - t0
    depth = synth.depth(1, cfg["height"], cfg["width"], synth.seed_for(cfg_idx, 3)).numpy()[0]
    t0 = time.perf_counter()
    orr.focus_map(frames[min(N - 1, 20)]["points"], cfg["width"], cfg["height"], orr.NORM_MAX, depth)
    t_render = time.perf_counter() - t0
    n_global = layers // 2 if layers > 1 else 1
    n_frame = layers - n_global
    total = Nw * (n_global * t_global * S / rows + n_frame * t_frame * W) + t_pose + N * t_render
    cores = len(os.sched_getaffinity(0))
    blas = max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    desc = (f"global attention: {rows} sampled query rows x {H} heads of 1 window ({t_global:.2f}s); frame attention: 1 frame x "
            f"{H} heads ({t_frame:.2f}s); pose chain + motion points: whole clip ({t_pose:.2f}s); Eq.7 render: 1 frame "
            f"{cfg['width']}x{cfg['height']} ({t_render:.2f}s); whole-clip seconds EXTRAPOLATED = {total:.0f}")
    return N / total, t_global + t_frame + t_pose + t_render, desc, min(cores, blas) if blas > 1 else 1


def dims_of(cfg_idx, args, num_windows):
    """num_windows: the caller's window count (the library's mf_num_windows for our arm, oracle/windows.py for the reference arm)."""
    from paper_2601_07154_b200 import synth
    c = synth.CONFIGS[cfg_idx]
    nw = num_windows(c["N"], c["W"], c["stride"])
    n = c["N"]
    if args.max_windows and args.max_windows < nw:
        nw = args.max_windows
        n = (nw - 1) * c["stride"] + c["W"]
    return dict(W=c["W"], P=c["P"], H=c["H"], D=c["D"], S=c["W"] * c["P"], Nw=nw, N=n, layers=c["layers"])


def config_block(cfg_idx, dims, args, extra=None):
    from paper_2601_07154_b200 import synth
    c = synth.CONFIGS[cfg_idx]
    d = {"workload": f"{'BASELINE.json configs[%d]' % cfg_idx if cfg_idx < 5 else 'extra workload (not in BASELINE.json)'} {c['name']}-shaped: W={dims['W']} stride={c['stride']} over "
                     f"{dims['N']} frames ({dims['Nw']} windows), P={dims['P']} tokens/frame, S={dims['S']}, "
                     f"{dims['layers']} alternating frame/global layers, H={dims['H']}, D={dims['D']}, bf16; "
                     f"focus map + guided depth at {c['width']}x{c['height']} fp32, N_points=15, sigma={c['sigma']}",
         "windows_per_launch": args.windows_per_launch, "focus_chunk_frames": args.focus_chunk,
         "l2": "inputs per step exceed L2 (no flush needed)"}
    if extra:
        d.update(extra)
    return d


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import windows as ow
    dims = dims_of(args.config, args, ow.num_windows)
    vals, secs, desc, cores = [], [], "", 1
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        fps, _, desc, cores = oracle_sample(args.config, dims, rows=256)
        if i >= args.warmup:
            vals.append(fps)
            secs.append(time.perf_counter() - t0)
    value = sum(vals) / len(vals)
    line = {"impl": "reference", "metric": "frames/sec at W=32 (window attention stack + pose chain + motion focus)",
            "value": value, "unit": "frames/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * sum(secs) / len(secs), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": config_block(args.config, dims, args),
            "cpu_baseline": {"value": value, "unit": "frames/s", "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": "frames/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def timed_steps(wl, steps, warmup, barrier, reduce_max, gpu_index):
    """W untimed + K timed passes of the whole hot path, bracketed by a barrier and CUDA events; clocks sampled meanwhile."""
    import torch
    for _ in range(warmup):
        wl.step_device()
    sampler = ClockSampler(gpu_index)
    ev_g, ev_f = [], []
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        wl.step_device(ev_g, ev_f)
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = reduce_max(e0.elapsed_time(e1))
    g_ms = sum(a.elapsed_time(b) for a, b, _ in ev_g)
    g_windows = sum(n for _, _, n in ev_g)
    f_ms = sum(a.elapsed_time(b) for a, b, _ in ev_f)
    f_frames = sum(n for _, _, n in ev_f)
    focus_gbs = 12.0 * f_frames * wl.width * wl.height / (f_ms * 1e-3) / 1e9 if f_ms > 0 else 0.0
    # Bytes the call has to move: M and G are written everywhere (8 B/pixel), D is read only where the map is non-zero
    # (reading G1: G = 0 wherever M = 0).  The render pass decides per warp (128 columns x one 32-row strip), so the share
    # of such blocks of the first chunk's maps that hold a non-zero pixel estimates the share of pixels whose depth is read.
    n = min(wl.chunk, wl.N)
    live = torch.nn.functional.max_pool2d((wl.fmap[:n] != 0).to(torch.float16).unsqueeze(1), kernel_size=(32, 128), ceil_mode=True)
    live_share = float(live.float().mean())
    return dict(ms_total=ms_total, ms_step=ms_total / steps, clocks=clocks, g_ms=g_ms, g_windows=g_windows, g_launches=len(ev_g),
                f_ms=f_ms, f_frames=f_frames,
                tflops=wl.flops_global * g_windows / (g_ms * 1e-3) / 1e12 if g_ms > 0 else 0.0,
                focus_gbs=focus_gbs, focus_live_share=live_share, focus_moved_gbs=focus_gbs * (8.0 + 4.0 * live_share) / 12.0)


def measure_windows_per_launch(wl, torch, api, peak_sustained, batches=(1, 2, 4, 8)):
    """the GLOBAL launch of this workload with 1, 2, 4 and 8 windows per launch, ~0.4 s of back-to-back launches each."""
    out = {}
    for b in batches:
        if b > wl.Nw:
            continue
        q, k, v = wl.q[:b], wl.k[:b], wl.v[:b]
        o = torch.empty_like(q)
        for _ in range(2):
            api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_GLOBAL, out=o)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_GLOBAL, out=o); e1.record()
        torch.cuda.synchronize()
        n = max(3, int(400.0 / max(e0.elapsed_time(e1), 1e-3)))
        e0.record()
        for _ in range(n):
            api.window_attention(q, k, v, wl.W, wl.P, api.ATTN_GLOBAL, out=o)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / n
        tf = wl.flops_global * b / (ms * 1e-3) / 1e12
        out[str(b)] = {"ms_per_launch": ms, "tflops": tf, "frac_of_sustained_peak": tf / peak_sustained}
    return out


def oracle_full_small(cfg_idx, dims):
    """SURVEY 8(d) procedure 4 for the two small configs: the oracle evaluated IN FULL, not on sampled rows -- the whole clip for
    the tiny config; one whole window (every row of one FRAME and one GLOBAL layer) for the suburban config, the clip's other
    windows and layers being repeats of the same work (stated as such).  Returns a cpu_baseline block."""
    import numpy as np
    from oracle import attention as oa
    from oracle import chain as oc
    from oracle import points as op
    from oracle import render as orr
    from oracle import windows as ow
    from paper_2601_07154_b200 import synth
    cfg = synth.CONFIGS[cfg_idx]
    W, P, H, D, S, Nw, N, layers = (dims[k] for k in ("W", "P", "H", "D", "S", "Nw", "N", "layers"))
    q, k, v = (t.float().numpy().astype(np.float64) for t in synth.qkv(1, S, H, D, synth.seed_for(cfg_idx, 0)))
    t0 = time.perf_counter()
    oa.window_attention(q, k, v, W, P, oa.GLOBAL)
    t_global = time.perf_counter() - t0
    t_frame = 0.0
    if layers > 1:
        t0 = time.perf_counter()
        oa.window_attention(q, k, v, W, P, oa.FRAME)
        t_frame = time.perf_counter() - t0
    traj = synth.trajectory(cfg, synth.seed_for(cfg_idx, 1), N)
    loc = synth.local_windows(traj, W, ow.window_starts(N, W, cfg["stride"]), seed=synth.seed_for(cfg_idx, 2), perturb_rot=1e-3, perturb_t=1e-3)
    t0 = time.perf_counter()
    poses = oc.chain_poses(loc.tolist(), W, cfg["stride"], N)
    frames = op.motion_points(poses, cfg["fx"], cfg["fy"], cfg["cx"], cfg["cy"], cfg["width"], cfg["height"], 15, cfg["sigma"])
    t_pose = time.perf_counter() - t0
    n_render = N if cfg_idx == 0 else 2
    depth = synth.depth(n_render, cfg["height"], cfg["width"], synth.seed_for(cfg_idx, 3)).numpy()
    t0 = time.perf_counter()
    for f in range(n_render):
        orr.focus_map(frames[N - 1 - f]["points"], cfg["width"], cfg["height"], orr.NORM_MAX, depth[f])
    t_render = (time.perf_counter() - t0) / n_render
    n_global = layers // 2 if layers > 1 else 1
    n_frame = layers - n_global
    total = Nw * (n_global * t_global + n_frame * t_frame) + t_pose + N * t_render
    whole = cfg_idx == 0
    return {"value": N / total, "unit": "frames/s", "kind": "oracle", "cores": len(os.sched_getaffinity(0)),
            "sample": ("whole clip evaluated in full" if whole else
                       f"one whole window evaluated in full (all {S} rows x {H} heads, one GLOBAL layer {t_global:.2f}s + one FRAME layer "
                       f"{t_frame:.2f}s), pose chain + motion points of the whole clip ({t_pose:.2f}s), Eq.7 render of {n_render} frames "
                       f"({t_render:.2f}s each); the other {Nw - 1} windows, {layers - 2} layers and {N - n_render} frames repeat this work: "
                       f"whole-clip seconds = {total:.0f}"),
            "seconds_measured": t_global + t_frame + t_pose + t_render * n_render}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    from paper_2601_07154_b200 import api, replicas
    rank, local_rank, world = replicas.env_world()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    replicas.init("nccl", dev)
    api.lib()
    peaks = measured_peaks()
    wl = Workload(args.config, args, dev)
    wl.setup_device()

    def barrier():
        replicas.barrier(dev)

    def reduce_max(x):
        return replicas.max_over_ranks(x, dev)

    res = timed_steps(wl, args.steps, args.warmup, barrier, reduce_max, local_rank)
    ms_total, ms_step, clocks = res["ms_total"], res["ms_step"], res["clocks"]
    value = replicas.whole_job_value(wl.N, ms_step, world)
    tflops, focus_gbs = res["tflops"], res["focus_gbs"]
    traffic = ncu_traffic(args.config, wl.B)
    roofline = {"bound": "tensor", "kernel": "window_attention_split_kernel (GLOBAL mode; the time is the whole mf_window_attention call: "
                                                   "key_norm_max_kernel, the pass over K for the score bound, runs ahead of it and window_attention_kernel, "
                                                   "for CTAs outside the bound, behind it on the same stream)", "achieved": tflops,
                "peak": peaks["tf_sustained"], "unit": "TFLOP/s", "frac": tflops / peaks["tf_sustained"],
                "peak_source": f"MEASURED_PEAKS.json bf16_tflops_sustained ({peaks['source']}); kernel timed inside a long step",
                "frac_of_burst": tflops / peaks["tf_burst"], "frac_of_nominal_2250": tflops / 2250.0,
                "flops_per_launch": wl.flops_global * wl.B, "ms_per_launch": res["g_ms"] / max(res["g_launches"], 1),
                "share_of_step": res["g_ms"] / ms_total, "traffic": traffic,
                "traffic_source": "NOT measured in this run: dram__bytes_read.sum + dram__bytes_write.sum of the committed `ncu --set full` "
                                  "capture of this launch shape (profiles/r2_ncu_attn.md, r2_ncu_attn_traffic.csv); algorithmic Q,K,V,O "
                                  f"bytes per launch = {8.0 * wl.S * wl.H * wl.D * wl.B:.0f}"}
    focus = {"bound": "hbm", "kernel": "mf_motion_focus (points+tables+norm+render, 12 B/pixel algorithmic: read D, write M, write G)",
             "achieved": focus_gbs, "peak": peaks["hbm"], "unit": "GB/s", "frac": focus_gbs / peaks["hbm"],
             "share_of_step": res["f_ms"] / ms_total,
             "bytes_moved": {"gbs": res["focus_moved_gbs"], "frac": res["focus_moved_gbs"] / peaks["hbm"],
                             "per_pixel": 8.0 + 4.0 * res["focus_live_share"], "depth_read_share": res["focus_live_share"]},
             "note": "`achieved` counts SURVEY 8(d)'s algorithmic 12 B/pixel (read D, write M, write G).  Since round 2 the call does not "
                     "read D where M is exactly zero (reading G1), so it MOVES fewer bytes: `bytes_moved` is the same time against "
                     "8 B/pixel + 4 B/pixel x the estimated share of pixels whose depth is read (ncu: profiles/r2_ncu_focus.md)"}

    e2e = None
    if not args.no_e2e:
        wl.setup_host()
        wl.step_host()
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 2))
        for _ in range(n_e2e):
            wl.step_host()
        barrier()
        sec = reduce_max((time.perf_counter() - t0) / n_e2e)
        e2e = {"value": world * wl.N / sec, "unit": "frames/s", "h2d_bytes_per_step": int(wl.h2d), "d2h_bytes_per_step": int(wl.d2h),
               "steps": n_e2e, "note": "mf_window_attention_host + mf_chain_and_focus_host on pinned host buffers, called from 4 host threads on 4 streams"}
        wl.release_host()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        dims = dims_of(args.config, args, api.num_windows)
        fps, secs, desc, cores = oracle_sample(args.config, dims)
        cpu = {"value": fps, "unit": "frames/s", "cores": cores, "kind": "oracle", "sample": desc, "sample_seconds": secs,
               "cpu_model": cpu_model(), "nproc": os.cpu_count()}

    block = None
    if rank == 0 and not args.no_block and wl.layers > 1:
        block = measure_block(wl, torch, api)

    d128 = None
    if rank == 0 and not args.no_d128 and wl.D == 64:
        d128 = measure_d128(wl, torch, api, peaks["tf_sustained"])

    exact = None
    if rank == 0 and not args.no_d128 and wl.D == 64 and (wl.S + 127) // 128 >= 32:
        exact = measure_exact_path(wl, torch, api, peaks["tf_sustained"])

    one_wave = None
    if rank == 0 and wl.S <= 2048:
        one_wave = measure_one_wave(wl, torch, api, peaks["tf_sustained"])

    streaming = None
    if rank == 0 and not args.no_stream and wl.Nw >= 8 and wl.layers > 1:
        streaming = measure_streaming(wl, torch, api)

    wpl = None
    if rank == 0 and world == 1 and wl.Nw >= 8 and wl.layers > 1:
        wpl = measure_windows_per_launch(wl, torch, api, peaks["tf_sustained"])

    # every BASELINE.json config in the driver-run line.  After the headline step, the other four configs run
    # 1 warm-up + 2 timed passes each (same step, same launch configuration), single GPU only.
    per_config = None
    launches_extra = 0
    if rank == 0 and world == 1 and args.config == 3 and not args.no_per_config and not args.max_windows:
        from paper_2601_07154_b200 import synth
        per_config = {synth.CONFIGS[3]["name"]: {"frames_per_s": value, "ms_per_step": ms_step, "global_tflops": tflops,
                                                 "frac_sustained": tflops / peaks["tf_sustained"], "focus_gbs": focus_gbs,
                                                 "focus_frac": focus_gbs / peaks["hbm"], "focus_moved_gbs": res["focus_moved_gbs"],
                                                 "focus_moved_frac": res["focus_moved_gbs"] / peaks["hbm"], "sm_mhz": clocks.get("sm_mhz"),
                                                 "steps": args.steps, "window_size": wl.W}}
        del wl
        torch.cuda.empty_cache()
        for ci in (0, 1, 2, 4):
            w2 = Workload(ci, args, dev)
            w2.setup_device()
            steps2 = 20 if ci == 0 else 2
            r2 = timed_steps(w2, steps2, 3 if ci < 2 else 1, barrier, reduce_max, local_rank)
            entry = {"frames_per_s": w2.N / (r2["ms_step"] * 1e-3), "ms_per_step": r2["ms_step"], "global_tflops": r2["tflops"],
                     "frac_sustained": r2["tflops"] / peaks["tf_sustained"], "focus_gbs": r2["focus_gbs"],
                     "focus_frac": r2["focus_gbs"] / peaks["hbm"], "focus_moved_gbs": r2["focus_moved_gbs"],
                     "focus_moved_frac": r2["focus_moved_gbs"] / peaks["hbm"], "sm_mhz": r2["clocks"].get("sm_mhz"),
                     "reasons": r2["clocks"].get("reasons"), "steps": steps2, "window_size": w2.W,
                     "workload": config_block(ci, dims_of(ci, args, api.num_windows), args)["workload"]}
            if ci == 0:
                entry["windows_148"] = measure_one_wave(w2, torch, api, peaks["tf_sustained"])
            if ci in (0, 1) and not args.no_cpu_baseline:
                entry["cpu_baseline"] = oracle_full_small(ci, dims_of(ci, args, api.num_windows))
            launches_extra += w2.launches * steps2
            per_config[synth.CONFIGS[ci]["name"]] = entry
            del w2
            torch.cuda.empty_cache()
        wl = None

    if rank == 0:
        dims = dims_of(args.config, args, api.num_windows)
        step_launches = Workload.launches_per_step(args.config, args, api)
        line = {"metric": "frames/sec at W=32 (window attention stack + pose chain + motion focus)", "value": value,
                "unit": "frames/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": config_block(args.config, dims, args), "parallelism": f"replicas x{world} (one clip per GPU)",
                "roofline": roofline, "focus_roofline": focus,
                "attention_tflops_all_layers": Workload.flops_per_step(args.config, args, api) * args.steps / (ms_total * 1e-3) / 1e12,
                "cpu_baseline": cpu, "e2e": e2e, "block": block, "head_dim_128": d128, "exact_path": exact, "windows_148": one_wave, "streaming": streaming,
                "windows_per_launch_sweep": wpl, "per_config": per_config,
                "gpu_launches": step_launches * args.steps, "gpu_launches_per_config_runs": launches_extra, "clocks": clocks}
        print(json.dumps(line))
    replicas.finish()


if __name__ == "__main__":
    main()
