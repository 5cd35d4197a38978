#!/usr/bin/env python
"""bench.py -- throughput of the L.A.Cosmic hot path on B200 (contract: see DESIGN.md section 7).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config2|config1|config0|stream]
    python bench.py --impl reference ...        # the CPU oracle on the host cores, same metric

One "step" = one whole pass of the hot path (all section-8(a) rows: niter = 4 iterations of steps
(1)-(7) plus frame prologue/epilogue) over one synthetic 4000x6500 fp32 frame (BASELINE.json
configs[2]).  `value` = frames/s with the frame resident in HBM (CUDA events around each step, L2
flushed between steps, max over ranks); `e2e` = the same through lacosmic_run_host with pinned HOST
buffers, H2D + D2H inside the timed region.  Frames are independent, so N GPUs run N replicas with
no collective ("scaling": "weak").  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2602_17938_b200 import replicas, synth  # noqa: E402

METRIC = "frames/s, 4000x6500 fp32 L.A.Cosmic (niter=4)"
# ALU-pipe roofline: FMNMX/FMNMX3 issue at 64 lanes/clk/SM (measured,
# profiles/r01_alu_minmax_microbench.txt) -> 148 SM x 64 x clocks.max.sm.
ALU_LANES_PER_CLK_SM = 64
N_SM = 148
# min/max (ALU-pipe FMNMX) instructions the dominant kernel executes per output pixel, from its SASS
# (DESIGN.md section 5 table; cross-checked against ncu smsp__inst_executed_pipe_alu in profiles/).
FINE_GATES_MINMAX_PER_PX = None   # filled from the library's own accounting below
# reference compare-exchanges per pixel per iteration with per-pixel networks:
REF_COMPARISONS_PER_PX_ITER = 19 + 99 + 99 + 480
# dram bytes per launch of the dominant kernel from the committed `ncu --set full` capture
# (profiles/; None until captured)
NCU_TRAFFIC_BYTES = {"fine_gates": 239900000,      # dense mode: profiles/r01_v9_ncu_full_dense.md
                     "noise_S": 269300000}         # lazy mode (with the work = img_in copy): profiles/r01_v9_ncu_full.md


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (profiling recipe's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu, self.proc, self.lines = gpu_index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
            t0 = time.time()
            while not self.lines and time.time() - t0 < 5.0:     # first sample before the timed region
                time.sleep(0.01)
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for nm, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return dict(sm_mhz=statistics.median(sm) if sm else None,
                    sm_max_mhz=max(smax) if smax else None,
                    power_w_max=max(power) if power else None,
                    samples=len(sm), reasons=sorted(reasons))


def _workload(name):
    if name == "config2":
        return dict(cfg=2, label="configs[2]: 4000x6500 fp32, 8000 stars, 30000 CRs, 0.5% salt-and-pepper")
    if name == "config1":
        return dict(cfg=1, label="configs[1]: 2048x2048 fp32")
    if name == "config0":
        return dict(cfg=0, label="configs[0]: 512x512 fp32")
    raise SystemExit("unknown workload " + name)


# ------------------------------------------------------------------------------------------- oracle legs
def _oracle_sample(img, params, rows, threads=None):
    """Time the oracle, as it stands, on the top `rows` rows of the frame (a bounded sample)."""
    from oracle import lacosmic_oracle as orc   # allowed here: cpu_baseline / --impl reference legs
    orc.build()
    crop = np.ascontiguousarray(img[:rows])
    allthreads = orc.max_threads()
    if threads:
        orc.set_threads(threads)
    t0 = time.perf_counter()
    orc.run(crop, **params)
    dt = time.perf_counter() - t0
    used = orc.max_threads()
    if threads:
        orc.set_threads(allthreads)
    return dt, crop.size, used


def run_reference(args):
    rank, _, _ = replicas.env_rank_world()
    if rank != 0:                            # under torchrun rank 0 alone runs the oracle; the others exit 0
        return 0
    wl = _workload(args.workload)
    frame = synth.make_config(wl["cfg"])
    params = dict(synth.DEFAULT_PARAMS)
    h, w = frame.img.shape
    rows = min(h, max(64, h // 8))          # 1/8 of the frame per step: a few seconds per step
    times = []
    for i in range(args.warmup + args.steps):
        dt, px, cores = _oracle_sample(frame.img, params, rows)
        if i >= args.warmup:
            times.append(dt)
    per_frame = statistics.mean(times) * (h * w) / px
    value = 1.0 / per_frame
    sample = "top %d of %d rows of the frame per step, time scaled by pixel count" % (rows, h)
    line = dict(impl="reference", metric=METRIC, value=value, unit="frames/s", n_gpus=args.gpus,
                steps=args.steps, warmup=args.warmup, ms_per_step=per_frame * 1e3,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
                config=dict(workload=wl["label"], h=h, w=w, niter=params["niter"], sigclip=params["sigclip"],
                            sigfrac=params["sigfrac"], objlim=params["objlim"],
                            parallelism="rank 0 only (the oracle on the host cores)"),
                mpix_per_s=value * h * w / 1e6,
                cpu_baseline=dict(value=value, unit="frames/s", cores=cores, kind="oracle", sample=sample),
                e2e=dict(value=value, unit="frames/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------- CUDA arm
def run_cuda(args):
    import torch
    import torch.distributed as dist

    import paper_2602_17938_b200 as lc

    rank, local_rank, world = replicas.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    lc.load_library()
    peaks = _peaks()

    wl = _workload(args.workload)
    # replicas: every rank cleans its own frame (same generator, seed offset by rank)
    kw = dict(synth.CONFIGS[wl["cfg"]])
    kw["seed"] = replicas.rank_seed(kw["seed"], rank)
    frame = synth.make_frame(**kw)
    params = dict(synth.DEFAULT_PARAMS)
    modes = {"lazy": lc.MODE_LAZY, "dense": lc.MODE_DENSE}
    P = {m: lc.Params(mode=v, **params) for m, v in modes.items()}
    h, w = frame.img.shape
    npx = h * w

    img = torch.from_numpy(frame.img).to(dev)
    mask = torch.empty((h, w), dtype=torch.uint8, device=dev)
    clean = torch.empty_like(img)
    ws = torch.empty(lc.lacosmic_workspace_bytes(h, w), dtype=torch.uint8, device=dev)
    counts = torch.zeros(params["niter"], dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2
    stream = torch.cuda.current_stream()

    def make_step(mode):
        def step():
            lc.lacosmic_run_ws(img, P[mode], mask_out=mask, clean_out=clean, workspace=ws, iter_counts=counts)
        return step

    def barrier():
        replicas.barrier(world, torch.cuda.synchronize)

    def timed(fn, steps, warmup):
        for _ in range(warmup):
            fn()
        barrier()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
               for _ in range(steps)]
        for a, b in evs:
            flush.zero_()                    # L2 flush, outside the event pair
            a.record(stream)
            fn()
            b.record(stream)
        barrier()
        per_step = [a.elapsed_time(b) for a, b in evs]
        timed.last = dict(median=statistics.median(per_step), min=min(per_step), max=max(per_step))   # this rank
        total_ms = replicas.max_over_ranks(sum(per_step), world, dev)
        return total_ms / steps

    def measure(mode):
        """value leg: K timed steps with the library's per-kernel event spans, then the same without."""
        step = make_step(mode)
        lc.lacosmic_kernel_timing_enable(True)
        for _ in range(args.warmup):
            step()
        torch.cuda.synchronize()
        lc.lacosmic_kernel_timing_read()         # drop warm-up spans
        ms = timed(step, args.steps, 0)
        kt = lc.lacosmic_kernel_timing_read()
        lc.lacosmic_kernel_timing_enable(False)
        launches = lc.lacosmic_last_launch_count()
        ms_nospans = timed(step, args.steps, 1)
        spread = dict(timed.last)
        # `ms` (the headline) is the run WITHOUT the library's per-kernel event pairs (34 extra event records per
        # step cost ~0.1 ms); the per-kernel durations come from the identical K steps timed with them
        return dict(ms=ms_nospans, ms_spans=ms, spread=spread, kt=kt, launches=launches,
                    counts=counts.cpu().numpy().tolist(), mask=mask.clone(), clean=clean.clone())

    # ---- device-resident timing (value): the production path, then the dense reference path
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    main_mode = args.mode
    other_mode = "dense" if main_mode == "lazy" else "lazy"
    res = measure(main_mode)
    res_other = measure(other_mode)
    modes_agree = bool(torch.equal(res["mask"], res_other["mask"]) and torch.equal(res["clean"], res_other["clean"])
                       and res["counts"] == res_other["counts"])
    mask_frac = float(res["mask"].float().mean().item())

    # ---- the same frame with no gain supplied (estimated at each iteration, R21)
    gain_est = None
    if not args.no_gain_estimation:
        pe = lc.Params(mode=modes[main_mode], **dict(params, gain=0.0))
        gains_t = torch.zeros(params["niter"], dtype=torch.float32, device=dev)

        def step_est():
            return lc.lacosmic_run_ws(img, pe, mask_out=mask, clean_out=clean, workspace=ws, iter_counts=counts)
        lc.lacosmic_kernel_timing_enable(True)
        step_est()
        torch.cuda.synchronize()
        lc.lacosmic_kernel_timing_read()
        ms_est = timed(step_est, max(3, args.steps // 2), 1)
        kt_est = lc.lacosmic_kernel_timing_read()
        lc.lacosmic_kernel_timing_enable(False)
        ge = lc.lacosmic_run_ws(img, pe, mask_out=mask, clean_out=clean, workspace=ws, iter_counts=counts,
                                want_gains=True)
        torch.cuda.synchronize()
        nsel = max(kt_est["gain_select"][1], 1)
        # one estimate = 18 histogram passes over the residual plane (4 B/px) + 3 over residual and med5 (8 B/px)
        sel_ms = kt_est["gain_select"][0] / nsel
        gain_est = dict(frames_per_s=world * 1e3 / ms_est, ms_per_step=ms_est,
                        gains=[float(v) for v in ge["gains"].cpu().numpy()],
                        new_cr_per_iteration=counts.cpu().numpy().tolist(),
                        select_ms_per_estimate=sel_ms,
                        select_hbm_gbs=96 * npx / (sel_ms * 1e-3) / 1e9,
                        select_hbm_frac=96 * npx / (sel_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                        note="gain = 0: residual plane + (3 rounds x 2 + 1) selections x 3 radix passes per iteration, "
                             "then every plane recomputed with the estimated gain (no incremental iterations)")

    # ---- configs[3] in small: a stream of independent frames with per-frame parameters, resident in HBM,
    # through lacosmic_run_batch, back to back (concurrency 1) and with several frames in flight
    stream_res = None
    if args.stream_frames > 0 and main_mode == "lazy":
        nf = args.stream_frames
        cfg = synth.stream_config(nf)
        imgs = torch.empty((nf, h, w), dtype=torch.float32, device=dev)
        for j, (kwj, _) in enumerate(cfg):
            kwj = dict(kwj)
            kwj["seed"] = replicas.rank_seed(kwj["seed"], rank)
            imgs[j].copy_(torch.from_numpy(synth.make_frame(**kwj).img))
        plist = [lc.Params(mode=lc.MODE_LAZY, **pj) for _, pj in cfg]
        masks = torch.empty((nf, h, w), dtype=torch.uint8, device=dev)
        cleans = torch.empty_like(imgs)
        bcounts = torch.zeros((nf, lc.MAX_NITER), dtype=torch.int32, device=dev)
        stream_res = dict(frames=nf, workload="configs[3] generator (seeds 1000.., sigclip cycling 4.0/4.5/5.0), "
                                             "%d frames resident in HBM" % nf)
        ref_out = None
        for kc in (1, args.stream_concurrency):
            bws = torch.empty(lc.lacosmic_batch_workspace_bytes(h, w, kc), dtype=torch.uint8, device=dev)

            def step_batch():
                lc.lacosmic_run_batch(imgs, plist, masks_out=masks, cleans_out=cleans, workspace=bws,
                                      iter_counts=bcounts)
            ms_b = timed(step_batch, 3, 1)
            out = (masks.clone(), cleans.clone())
            if ref_out is None:
                ref_out = out
            else:
                stream_res["same_as_back_to_back"] = bool(torch.equal(out[0], ref_out[0]) and
                                                          torch.equal(out[1], ref_out[1]))
            stream_res["concurrency_%d" % kc] = dict(frames_per_s=world * nf * 1e3 / ms_b, ms_per_frame=ms_b / nf)
            del bws
        del imgs, masks, cleans, ref_out, out
        torch.cuda.empty_cache()

    # ---- end to end through the host-buffer C-ABI call
    img_h = torch.from_numpy(frame.img).pin_memory()
    mask_h = torch.empty((h, w), dtype=torch.uint8).pin_memory()
    clean_h = torch.empty((h, w), dtype=torch.float32).pin_memory()
    hws = torch.empty(lc.lacosmic_host_workspace_bytes(h, w), dtype=torch.uint8, device=dev)

    def step_host():
        lc.lacosmic_run_host(img_h, P[main_mode], mask_out_host=mask_h, clean_out_host=clean_h, dev_workspace=hws)

    ms_e2e = timed(step_host, args.steps, max(1, args.warmup // 2))
    same = bool((mask_h.numpy() == res["mask"].cpu().numpy()).all() and
                (clean_h.numpy() == res["clean"].cpu().numpy()).all())
    # ---- raw uint16 ingest: the same frame rounded to detector counts, 2 bytes per pixel H2D
    raw_h = torch.from_numpy(np.clip(np.rint(frame.img), 0, 65535).astype(np.uint16)).pin_memory()

    def step_host_u16():
        lc.lacosmic_run_host(raw_h, P[main_mode], mask_out_host=mask_h, clean_out_host=clean_h, dev_workspace=hws)
    ms_u16 = timed(step_host_u16, max(3, args.steps // 2), 1)
    e2e_u16 = dict(value=world * 1e3 / ms_u16, unit="frames/s", ms_per_step=ms_u16, h2d_bytes_per_step=npx * 2,
                   d2h_bytes_per_step=npx * 5, call="lacosmic_run_host_u16 (pinned host buffers, uint16 input)",
                   note="input = the bench frame rounded to uint16 counts: a different input, reported beside e2e")
    # ---- sparse results: bit-plane mask + list of replaced pixels instead of the two full planes over PCIe
    sp_out = lc.lacosmic_run_host_sparse(img_h, P[main_mode], capacity=npx // 32, dev_workspace=hws)
    torch.cuda.synchronize()

    def step_host_sparse():
        lc.lacosmic_run_host_sparse(img_h, P[main_mode], out=sp_out, dev_workspace=hws)
    ms_sp = timed(step_host_sparse, max(3, args.steps // 2), 1)
    nsp = int(sp_out["count"][0])
    sp_idx = sp_out["idx"].numpy()[:nsp]
    sp_ok = bool(nsp == int(res["mask"].sum().item()) and nsp <= sp_out["capacity"] and
                 (sp_out["val"].numpy()[:nsp] == res["clean"].cpu().numpy().ravel()[sp_idx]).all())
    e2e_sparse = dict(value=world * 1e3 / ms_sp, unit="frames/s", ms_per_step=ms_sp, h2d_bytes_per_step=npx * 4,
                      d2h_bytes_per_step=int(sp_out["maskbits"].numel() * 4 + 8 * sp_out["capacity"] + 4),
                      flagged=nsp, capacity=int(sp_out["capacity"]), matches_device_path=sp_ok,
                      call="lacosmic_run_host_sparse (pinned host buffers; outputs: bit-plane mask + ascending "
                           "list of flagged pixels with their replacement values)")
    step_host()                                  # leave the fp32 results in mask_h / clean_h for the checks below
    torch.cuda.synchronize()

    # ---- end to end on a stream of frames: lacosmic_run_host_batch overlaps the H2D copy of one frame, the
    # kernels of another and the D2H copy of a third
    e2e_stream = None
    if args.stream_frames > 0:
        nh = min(args.stream_frames, 8)
        imgs_h = torch.empty((nh, h, w), dtype=torch.float32).pin_memory()
        for j in range(nh):
            imgs_h[j].copy_(img_h)                     # the bench frame, nh times: timing only
        masks_h = torch.empty((nh, h, w), dtype=torch.uint8).pin_memory()
        cleans_h = torch.empty((nh, h, w), dtype=torch.float32).pin_memory()
        kslots = 3
        hbws = torch.empty(lc.lacosmic_host_batch_workspace_bytes(h, w, kslots), dtype=torch.uint8, device=dev)
        plist_h = [P[main_mode]] * nh

        def step_host_batch():
            lc.lacosmic_run_host_batch(imgs_h, plist_h, masks_host=masks_h, cleans_host=cleans_h,
                                       dev_workspace=hbws)
        ms_hb = timed(step_host_batch, 3, 1)
        ok_hb = bool((masks_h[nh - 1].numpy() == mask_h.numpy()).all() and
                     (cleans_h[nh - 1].numpy() == clean_h.numpy()).all())
        e2e_stream = dict(value=world * nh * 1e3 / ms_hb, unit="frames/s", frames=nh, slots=kslots,
                          ms_per_frame=ms_hb / nh, h2d_bytes_per_frame=npx * 4, d2h_bytes_per_frame=npx * 5,
                          matches_single_frame_call=ok_hb,
                          call="lacosmic_run_host_batch (pinned host buffers, %d staging slots)" % kslots)
        # the production configuration: raw uint16 frames in, sparse results out (2 B/px in, ~0.4 B/px out)
        del masks_h, cleans_h
        prod = {}
        for name, src in (("f32", imgs_h), ("u16", None)):
            if src is None:
                src = torch.empty((nh, h, w), dtype=torch.uint16).pin_memory()
                for j in range(nh):
                    src[j].copy_(raw_h)
            sp_stream = lc.lacosmic_run_host_stream_sparse(src, plist_h, capacity=npx // 32, dev_workspace=hbws)
            torch.cuda.synchronize()

            def step_stream_sparse():
                lc.lacosmic_run_host_stream_sparse(src, plist_h, out=sp_stream, dev_workspace=hbws)
            ms_ss = timed(step_stream_sparse, 3, 1)
            prod[name] = dict(value=world * nh * 1e3 / ms_ss, unit="frames/s", ms_per_frame=ms_ss / nh,
                              h2d_bytes_per_frame=npx * (4 if name == "f32" else 2),
                              d2h_bytes_per_frame=int(sp_stream["maskbits"][0].numel() * 4 + 8 * sp_stream["capacity"] + 4),
                              flagged_per_frame=int(sp_stream["count"][nh - 1]))
            del sp_stream
        e2e_stream["sparse_results"] = dict(call="lacosmic_run_host_stream_sparse (%d frames, %d staging slots)" % (nh, kslots),
                                            **prod)
        del imgs_h, hbws, src
    clocks = sampler.stop() if rank == 0 else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    niter = params["niter"]
    sm_max = (clocks or {}).get("sm_max_mhz") or peaks["sm_max_mhz"]
    alu_peak = N_SM * ALU_LANES_PER_CLK_SM * sm_max * 1e6 / 1e12          # T min/max instr / s

    def summarise(r):
        kt = r["kt"]
        whole = max(kt["whole_frame"][0], 1e-9)
        return dict(frames_per_s=world * 1e3 / r["ms"], ms_per_step=r["ms"],
                    ms_per_step_with_kernel_event_spans=r["ms_spans"], launches_per_step=r["launches"],
                    kernels_ms_per_step={k: round(v[0] / args.steps, 4) for k, v in kt.items() if v[1]},
                    kernel_share_of_step={k: round(v[0] / whole, 4) for k, v in kt.items()
                                          if k != "whole_frame" and v[1]})

    def roofline(r):
        """ALU roofline of the class with the largest summed time."""
        kt = r["kt"]
        # dominant kernel = the launch that takes longest (classes whose launches all process the full
        # frame: their algorithmic work per launch is pixels x the per-pixel figure)
        dom = max((k for k in kt if k in KERNEL_MINMAX_PER_PX and kt[k][1]),
                  key=lambda k: kt[k][0] / kt[k][1])
        dom_ms, dom_spans = kt[dom]
        dom_avg_ms = dom_ms / max(dom_spans, 1)
        ops_px = KERNEL_MINMAX_PER_PX[dom]
        achieved = npx * ops_px / (dom_avg_ms * 1e-3) / 1e12
        return dict(bound="alu", kernel=dom, achieved=achieved, peak=alu_peak, unit="T min/max instr/s",
                    frac=achieved / alu_peak, traffic=(NCU_TRAFFIC_BYTES or {}).get(dom),
                    peak_source="148 SM x 64 ALU lanes/clk x %.0f MHz (DESIGN.md section 5; lanes/clk "
                                "measured in profiles/r01_alu_minmax_microbench.txt)" % sm_max,
                    minmax_instr_per_px=ops_px, avg_launch_ms=dom_avg_ms, launches_timed=dom_spans)

    frames_per_s = world * 1e3 / res["ms"]
    e2e_fps = world * 1e3 / ms_e2e
    bytes_iter = HBM_BYTES_PER_PX_ITER[main_mode]
    hbm_bytes_step = npx * (bytes_iter * niter + HBM_BYTES_PER_PX_FRAME)
    hbm = dict(algorithmic_bytes_per_step=hbm_bytes_step,
               achieved_gbs=hbm_bytes_step / (res["ms"] * 1e-3) / 1e9,
               peak_gbs=peaks["hbm_gbs"], peak_source=peaks["source"],
               frac=hbm_bytes_step / (res["ms"] * 1e-3) / 1e9 / peaks["hbm_gbs"])
    ref_cmp_rate = npx * REF_COMPARISONS_PER_PX_ITER * niter / (res["ms"] * 1e-3) / 1e12

    # ---- the oracle on the host cores: a bounded sample of the same frame
    cpu = None
    if not args.no_cpu_baseline:
        rows = min(h, 1000)
        dt, px, cores = _oracle_sample(frame.img, params, rows)
        cpu = dict(value=(px / npx) / dt, unit="frames/s", cores=cores, kind="oracle",
                   sample="top %d of %d rows of the same frame, one run, %.1f s; frames/s scaled by "
                          "pixel count" % (rows, h, dt))
        rows1 = min(h, 100)                      # also one thread, on a smaller sample
        dt1, px1, c1 = _oracle_sample(frame.img, params, rows1, threads=1)
        cpu["single_thread"] = dict(value=(px1 / npx) / dt1, unit="frames/s", cores=c1,
                                    sample="top %d rows, one run, %.1f s" % (rows1, dt1))

    main_sum = summarise(res)
    line = dict(
        metric=METRIC, value=frames_per_s, unit="frames/s", n_gpus=world, steps=args.steps,
        warmup=args.warmup, ms_per_step=res["ms"], higher_is_better=True, scaling="weak",
        vs_baseline=None, dtype="f32", data="synthetic",
        config=dict(workload=wl["label"], h=h, w=w, niter=niter, sigclip=params["sigclip"],
                    sigfrac=params["sigfrac"], objlim=params["objlim"], mode=main_mode,
                    l2="flushed between steps (256 MiB write outside the event pair)",
                    parallelism="replicas (one frame per GPU, no collective)"),
        mpix_per_s=frames_per_s * npx / 1e6,
        e2e=dict(value=e2e_fps, unit="frames/s", h2d_bytes_per_step=npx * 4,
                 d2h_bytes_per_step=npx * 5, ms_per_step=ms_e2e, matches_device_path=same,
                 call="lacosmic_run_host (pinned host buffers)"),
        gpu_launches=res["launches"] * args.steps,
        launches_per_step=res["launches"],
        roofline=roofline(res), hbm=hbm,
        kernels_ms_per_step=main_sum["kernels_ms_per_step"],
        kernel_share_of_step=main_sum["kernel_share_of_step"],
        ms_per_step_with_kernel_event_spans=res["ms_spans"],
        ms_per_step_spread={k: round(v, 4) for k, v in res["spread"].items()},
        ref_comparisons_T_per_s=ref_cmp_rate,
        other_mode=dict(mode=other_mode, same_mask_clean_counts=modes_agree, roofline=roofline(res_other),
                        **summarise(res_other)),
        stream=stream_res, e2e_stream=e2e_stream, e2e_u16=e2e_u16, e2e_sparse=e2e_sparse, gain_estimation=gain_est,
        new_cr_per_iteration=res["counts"], mask_fraction=mask_frac,
        clocks=clocks, cpu_baseline=cpu,
        context="paper (PAPER.md:31,47): 55 s/frame dfcosmic C++ at 2 threads on AWS; GPU variant on an "
                "RTX 5060 Ti >10x faster than CPU variants (no absolute number in the text)",
    )
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


# ALU-pipe min/max instructions per output pixel of each kernel class (static SASS
# count of FMNMX/FMNMX3 per pixel, halo recomputation included) -- the per-unit figure behind
# roofline.achieved.
KERNEL_MINMAX_PER_PX = {
    # generated networks (median_networks.cuh): med7 764/4, med5 326/4, med3 76/4 x 1.46 (haloed m3 tile)
    "fine_gates": 764 / 4 + 326 / 4 + 1.46 * 76 / 4,
    "noise_S": 326 / 4 + 13 / 4,                     # med5 + the clamp/floor selects of L+ and N
}
# HBM bytes per pixel per iteration the path must move with the current fusion:
# noise_S: read work 4 + write S 4; dense fine_gates: read work 4 + S 4 + 0.375 bit-planes; lazy: A1/A2
# bit-planes 0.25 + list passes ~1; dilate/replace ~1
HBM_BYTES_PER_PX_ITER = {"dense": 4 + 4 + 4 + 4 + 0.375 + 1.0, "lazy": 4 + 4 + 0.25 + 1.0 + 1.0}
HBM_BYTES_PER_PX_FRAME = 8 + 1.125


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="config2", choices=["config2", "config1", "config0"])
    ap.add_argument("--mode", default="lazy", choices=["lazy", "dense"],
                    help="which evaluation mode is the headline (the other is measured and reported too)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-gain-estimation", action="store_true", help="skip the gain = 0 leg (DESIGN.md R21)")
    ap.add_argument("--stream-frames", type=int, default=12,
                    help="frames of the configs[3] stream leg (0 = skip; 64 = the full configuration)")
    ap.add_argument("--stream-concurrency", type=int, default=4,
                    help="frames in flight in the stream leg (lacosmic_run_batch internal streams)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3                          # timing rule: at least 3 warm-up steps
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
