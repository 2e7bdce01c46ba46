"""bench.py — probe positions/s for one full forward+adjoint iteration of the multislice hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 3]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
           bench.py --gpus N --steps K --warmup W

A step = one pass of the whole hot path over ALL positions of the workload:
ptycho_gradient (loss + object / probe / position gradients) then ptycho_apply_update (SGD), through the C ABI.
Workload at N=1: BASELINE.json config 3 (128x128 patterns, 64x64 scan = 4096 positions, 8 modes, 20 slices, tilt,
Poisson loss), the configuration north_star's target is quoted on.  Inputs are seeded and synthetic.
After the headline workload the default invocation also times, briefly, configs 1, 2, 4, 5 (batch 1024) and the band-limited
variant of config 3 and attaches them as "secondary" (--no-secondary skips them).  Rank 0 prints ONE JSON line.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "probe positions/s per full forward+adjoint iteration"
UNIT = "positions/s"
PAPER_CONTEXT = "paper: <3 s/iter for 6400 positions x 20 slices on an RTX 3080, whole engine iteration (PAPER.md:266) - context only"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--cpu-sample", type=int, default=0, help="positions in the oracle sample (0: per-config default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--batch", type=int, default=0, help="config 5: mini-batch size of the LSQML sweep (0: sweep 64/256/1024/4096)")
    ap.add_argument("--bandlimit", type=float, default=0.0, help="timed variant: sharp band-limit mask at this fraction of Nyquist "
                    "inside the propagator (PAPER.md:117, reading R9); 0 = off, as in BASELINE.json's configs")
    ap.add_argument("--ws-gib", type=float, default=0.0, help="cap of the device workspace in GiB (0: library default)")
    ap.add_argument("--stash-fp16", action="store_true", help="timed variant: PT_STASH_FP16, the slice-wave stash stored as binary16 "
                    "pairs (SURVEY 8(f) rank 4; grad_object then within 7.5e-5 of the oracle instead of 3.4e-5, DESIGN.md 10)")
    ap.add_argument("--no-secondary", action="store_true", help="config 3 only: skip the short runs of the other configurations")
    return ap.parse_args()


def workload(idx, bandlimit=0.0):
    from paper_2505_14372_b200 import synth
    cfg = synth.config(idx) if bandlimit <= 0 else synth.config(idx, bandlimit=bandlimit)
    return cfg, dict(**({} if bandlimit <= 0 else {"variant": f"band-limited propagator, {bandlimit:g} x Nyquist"}), **dict(workload=f"BASELINE.json configs[{idx - 1}] ({cfg.name})", n=cfg.n, positions_per_gpu=cfg.n_pos, modes=cfg.n_modes,
                     slices=cfg.n_slices, object_px=cfg.obj_n, loss="poisson" if cfg.loss == synth.LOSS_POISSON else "amplitude",
                     start_state="O = exp((i-0.05) 0.8 phi_true), true probe, nominal positions",
                     patterns="seeded closed-form stand-in + Poisson (synth.standin_patterns)"))


def problem_kwargs(cfg):
    return dict(n=cfg.n, n_modes=cfg.n_modes, n_slices=cfg.n_slices, obj_ny=cfg.obj_n, obj_nx=cfg.obj_n,
                pixel_size=cfg.pixel_size, wavelength=cfg.wavelength, slice_thickness=[cfg.dz] * cfg.n_slices,
                tilt_x_mrad=cfg.tilt_mrad[0], tilt_y_mrad=cfg.tilt_mrad[1], bandlimit=cfg.bandlimit, loss=cfg.loss,
                loss_c=cfg.loss_c, eps=cfg.eps)


def host_inputs(cfg, rows=None):
    from paper_2505_14372_b200 import synth
    phi = synth.object_phase(cfg)
    obj = synth.object_from_phase(phi, 0.8)
    pr = synth.probe(cfg)
    pos = synth.positions(cfg)
    if rows is not None:
        pos = pos[rows]
    if rows is None and cfg.n_pos > UNIQUE_PATTERN_ROWS:
        # config 4 (16384 x 256 x 256 floats): draw UNIQUE_PATTERN_ROWS stand-in patterns and repeat them over the scan;
        # the work per position does not depend on the pattern values (no data-dependent branches)
        inten = np.tile(synth.standin_patterns(cfg, np.arange(UNIQUE_PATTERN_ROWS)), (cfg.n_pos // UNIQUE_PATTERN_ROWS, 1, 1))
    else:
        inten = synth.standin_patterns(cfg, rows)
    return obj, pr, pos, inten


UNIQUE_PATTERN_ROWS = 1024
MINIBATCH = {4: 1024}                                  # BASELINE.json configs[3]: mini-batches of 1024 positions
LR = dict(lr_obj=1e-7, lr_probe=1e-7, lr_pos=1e-9)   # a real (tiny) SGD step so every timed step does the update


# ----------------------------------------------------------------------------------------------------
# clocks during the timed region (profiling recipe)
# ----------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                       "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close(); os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", 1965.0


# per-position ALGORITHMIC bytes of the two FFT-chain kernels: the slice-wave stash of the
# reverse-mode adjoint (written once by k_forward, read once by k_backward: SURVEY §8(d) B_act) plus the
# far-field hand-over; the per-mode patch-gradient staging of the current build is NOT algorithmic.
def algorithmic_bytes_per_position(cfg, kernel):
    NN = cfg.n * cfg.n
    stash = cfg.n_modes * cfg.n_slices * NN * 8
    far = cfg.n_modes * NN * 8
    if kernel == "k_forward":
        return stash + far
    if kernel == "k_backward":
        return stash + far + NN * 4
    return None


def nominal_flops_per_position(cfg):
    NN = cfg.n * cfg.n
    fft = 5.0 * NN * np.log2(NN)                      # one 2-D complex FFT
    return cfg.n_modes * (4 * cfg.n_slices * fft + (32 * cfg.n_slices + 20) * NN)


# ----------------------------------------------------------------------------------------------------
def run_reference(args):
    """The reference arm of this tier = the CPU oracle as it stands, on the host cores, on a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    cfg, conf = workload(args.config, args.bandlimit)
    n = args.cpu_sample or {1: 256, 2: 64, 3: 16, 4: 4, 5: 16}[args.config]
    rows = np.arange(n)
    obj, pr, pos, inten = host_inputs(cfg, rows)
    pbo = orc.Problem(**problem_kwargs(cfg))

    def step():
        g = orc.gradient(pbo, obj, pr, pos, inten)
        orc.apply_update(pbo, 0, obj, pr, pos, g["grad_object"], g["grad_probe"], g["grad_pos"], **LR)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    v = n / dt
    sample = f"first {n} positions of the scan, forward+adjoint+SGD update per step"
    conf.update(sample_positions=n)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": conf,
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


def measure(args, cfg_idx, *, steps, warmup, dist, rank, world, local, bandlimit=0.0, batch=0, want_e2e=True, want_cpu=True,
            min_seconds=0.0, want_sweep=True, prof_steps=None):
    """One workload through the C ABI: K timed steps (CUDA events on the launching stream, clocks sampled meanwhile), then the
    per-kernel device times over the same steps, the host-buffer end-to-end loop and the oracle sample.  Returns a dict."""
    import torch
    from paper_2505_14372_b200 import ptycho, shard
    from paper_2505_14372_b200 import synth as _synth
    cfg, conf = workload(cfg_idx, bandlimit)
    J = cfg.n_pos
    obj_h, pr_h, pos_h, I_h = host_inputs(cfg)
    pbg = ptycho.Problem(**problem_kwargs(cfg))
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    obj, pr, pos, inten = dev(obj_h), dev(pr_h), dev(pos_h), dev(I_h)
    gO, gP = torch.empty_like(obj), torch.empty_like(pr)
    gX = torch.empty((J, 2), dtype=torch.float32, device="cuda")
    loss = torch.zeros(1, dtype=torch.float64, device="cuda")
    cap = int(args.ws_gib * (1 << 30)) if args.ws_gib > 0 else None
    mb = MINIBATCH.get(cfg_idx)
    lsqml = cfg_idx == 5
    if lsqml:
        mb = batch or 1024
    batches = None if mb is None else [torch.from_numpy(b).cuda() for b in _synth.batches(cfg, mb)]
    fl = ptycho.WANT_POS_GRAD | ((ptycho.WANT_ILLUM | ptycho.WANT_STEP_SIZES) if lsqml else 0)
    xfl = ptycho.STASH_FP16 if args.stash_fp16 else 0
    fl |= xfl
    if xfl:
        conf.update(variant="PT_STASH_FP16: slice-wave stash stored as binary16 pairs")
        want_e2e = False
    ws = ptycho.make_workspace(pbg, J, J if lsqml else (mb or J), fl, max_bytes=cap)
    if batches is not None and not lsqml:
        conf.update(minibatch=mb, grouping="seeded permutation (sparse), gradients accumulated over the batches, one update")
        want_e2e = False        # the host-buffer entry point takes one batch per call: no whole-iteration e2e at this size
    if lsqml:
        # config 5: per batch, gradient + illumination map + step-size sweep (second pass over the chain) + LSQML update
        conf.update(minibatch=mb, grouping="seeded permutation (sparse); per batch: gradient, step-size sweep, LSQML update",
                    flags="POS_GRAD | ILLUM | STEP_SIZES")
        illum = torch.zeros(obj.shape, dtype=torch.float32, device="cuda")
        illum_prev = torch.full(obj.shape, float(cfg.dose) / (cfg.step_px ** 2), dtype=torch.float32, device="cuda")   # ~ dose per scan-step area
        want_e2e = False        # the host-buffer entry point has no step-size outputs
        st_terms = torch.empty((J, 2 * cfg.n_slices + 6), dtype=torch.float32, device="cuda")
        LS = dict(mode=ptycho.UPDATE_LSQML, beta_obj=1e-3, beta_probe=1e-3, gamma=1e-2)

    def lsqml_iteration(bl):
        for b in bl:
            nb = b.numel()
            ptycho.gradient(pbg, obj, pr, pos, inten, b, workspace=ws, grad_object=gO, grad_probe=gP, grad_pos=gX[:nb], illum=illum,
                            illum_prev=illum_prev, step_terms=st_terms[:nb], loss=loss, flags=xfl)
            ptycho.apply_update(pbg, obj, pr, pos, grad_object=gO, grad_probe=gP, illum_prev=illum_prev, step_terms=st_terms[:nb],
                                batch_idx=b, workspace=ws, **LS)

    order = None if batches is None else torch.cat(batches)

    def step():
        # weak scaling over ranks: every rank owns J positions of the scan; object / probe are replicated, so the
        # only exchange is the sum of the object / probe gradients and the loss before the update.
        if lsqml:
            return lsqml_iteration(batches)
        if batches is None:
            ptycho.gradient(pbg, obj, pr, pos, inten, None, workspace=ws, grad_object=gO, grad_probe=gP, grad_pos=gX, loss=loss, flags=xfl)
        else:
            o = 0
            for i, b in enumerate(batches):
                ptycho.gradient(pbg, obj, pr, pos, inten, b, workspace=ws, grad_object=gO, grad_probe=gP,
                                grad_pos=gX[o:o + b.numel()], loss=loss, flags=(ptycho.ACCUMULATE if i else 0) | xfl)
                o += b.numel()
        if dist is not None:
            shard.allreduce_sums(dist, gO, gP, loss)
        if batches is None:
            ptycho.apply_update(pbg, obj, pr, pos, grad_object=gO, grad_probe=gP, grad_pos=gX, **LR)
        else:
            ptycho.apply_update(pbg, obj, pr, pos, grad_object=gO, grad_probe=gP, grad_pos=gX, batch_idx=order, **LR)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(warmup):
        step()
    assert ptycho.status(ws) == 0, "device-side error flag set during warm-up"
    if min_seconds > 0:
        # short workloads: enough steps for the timed region to last min_seconds, so that the 100 ms clock sampler sees it
        torch.cuda.synchronize(); e0.record(); step(); e1.record(); torch.cuda.synchronize()
        steps = max(steps, int(np.ceil(min_seconds * 1e3 / max(e0.elapsed_time(e1), 1e-3))))
    # timing rule: inputs larger than L2, or L2 flushed between timed iterations.  The per-step working set (patterns + stash +
    # staging + far fields) of configs 2-5 is far beyond the 126 MB L2; config 1's is not, so there every step is timed with
    # its own pair of events and a 512 MB buffer is overwritten between steps.
    wset = J * cfg.n * cfg.n * (4 + 8 * cfg.n_modes * (2 * cfg.n_slices + 2))
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda") if wset < 400e6 else None
    def time_steps(run):
        barrier()
        if flush is None:
            e0.record()
            for _ in range(steps):
                run()
            e1.record()
            barrier()
            return e0.elapsed_time(e1)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in evs:
            flush.zero_()
            a.record(); run(); b.record()
        barrier()
        return sum(a.elapsed_time(b) for a, b in evs)

    clocks = ClockSampler(local) if rank == 0 else None
    n0 = ptycho.launch_count()
    total_ms = time_steps(step)
    launches = ptycho.launch_count() - n0
    # Launch-bound workloads (single slice: a step is a dozen launches of a few microseconds each): the same step captured once
    # into a CUDA graph through the same C-ABI calls (the library allocates nothing and never synchronises, so it can be
    # captured) and replayed per timed step.  Every kernel runs again on every replay; only the host-side launch path differs.
    direct = None
    if cfg.n_slices == 1 and dist is None and not lsqml:
        graph = torch.cuda.CUDAGraph()
        n0 = ptycho.launch_count()
        with torch.cuda.graph(graph):
            step()
        per_step = ptycho.launch_count() - n0
        graph.replay()
        assert ptycho.status(ws) == 0, "device-side error flag set by the captured step"
        direct = {"value": world * J / (total_ms / steps * 1e-3), "unit": UNIT, "ms_per_step": total_ms / steps}
        total_ms = time_steps(graph.replay)
        launches = per_step * steps
        conf.update(launch="the step (ptycho_gradient + ptycho_apply_update) captured once in a CUDA graph (torch.cuda.CUDAGraph) and "
                           "replayed per timed step; `direct_call` is the same loop with one C-ABI call sequence per step")
    ms = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_step = ms.item() / steps
    clk = clocks.stop() if clocks else None
    loss_val = loss.item()
    assert np.isfinite(loss_val) and ptycho.status(ws) == 0

    sweep = None
    if lsqml and not batch and want_sweep:
        # the paper's grouping sweep: whole-iteration rate at each mini-batch size, one timed iteration each
        sweep = {str(mb): J / (ms_step * 1e-3)}
        for bsz in (64, 256, 4096):
            bl = [torch.from_numpy(b).cuda() for b in _synth.batches(cfg, bsz)]
            lsqml_iteration(bl)
            torch.cuda.synchronize(); e0.record(); lsqml_iteration(bl); e1.record(); torch.cuda.synchronize()
            sweep[str(bsz)] = J / (e0.elapsed_time(e1) * 1e-3)
        conf.update(batch_sweep_positions_per_s=sweep)

    # per-kernel device time (CUDA events on the launching stream, inside the library)
    psteps = min(steps, prof_steps) if prof_steps else steps
    ptycho.profile_enable(True)
    torch.cuda.synchronize()
    for _ in range(psteps):
        step()
    prof = ptycho.profile_read()
    ptycho.profile_enable(False)
    tot = sum(v[0] for v in prof.values())
    top = max(prof, key=lambda k: prof[k][0])
    top_ms, top_n = prof[top]
    hbm, which, sm_max = measured_peaks()
    units_per_launch = J * psteps / top_n
    ab = algorithmic_bytes_per_position(cfg, top)
    # The FFT chain kernels are bound by plain FP32 arithmetic (19.5 flop/B against a machine balance of
    # 11.4), so the line reports "alu": nominal FFT flops (5 N^2 log2 N^2 per 2-D FFT + pointwise) per launch over the
    # launch duration, against 148 SM x 128 lanes x 2 flop x max SM clock (peak) and against the FFMA rate measured on this
    # device in this run (peak_measured, ptycho_profile_fp32_peak).  The HBM view of the same kernel (algorithmic bytes:
    # stash + far field) is given beside it.
    fp32_peak = 148 * 128 * 2 * sm_max * 1e6 / 1e12
    fp32_meas = ptycho.profile_fp32_peak(ws)
    roof = {"bound": "alu", "kernel": top, "achieved": None, "peak": fp32_peak, "unit": "TFLOP/s", "frac": None, "traffic": None,
            "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 flop x sm_max_mhz (DESIGN.md §6)",
            "peak_measured": fp32_meas, "peak_measured_source": "FFMA micro-benchmark in this run (ptycho_profile_fp32_peak)",
            "share_of_step": top_ms / tot, "avg_launch_ms": top_ms / top_n,
            "kernel_ms_per_step": {k: v[0] / psteps for k, v in sorted(prof.items(), key=lambda kv: -kv[1][0])}}
    # flops of one launch of the dominant kernel: the forward and the backward chain each do half of the FFTs; the fused
    # single-slice kernel does all of them
    share = {"k_forward": 0.5, "k_backward": 0.5, "k_single": 1.0}.get(top)
    if share is not None:
        sec = top_ms / top_n * 1e-3
        fl = share * nominal_flops_per_position(cfg)
        ach = fl * units_per_launch / sec / 1e12
        roof.update(achieved=ach, frac=ach / fp32_peak, frac_of_measured_peak=ach / fp32_meas if fp32_meas > 0 else None,
                    nominal_flops_per_launch=fl * units_per_launch)
        if ab is not None:
            achb = ab * units_per_launch / sec / 1e9
            roof.update(hbm_view={"achieved": achb, "peak": hbm, "unit": "GB/s", "frac": achb / hbm, "peak_source": which,
                                  "algorithmic_bytes_per_launch": ab * units_per_launch})
    # traffic: DRAM bytes of one launch of that kernel from the committed `ncu --set full` capture (profiles/), scaled to
    # this run's positions per launch; null if the capture is of another kernel or workload
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", TRAFFIC_FILE)) as f:
            for tr in csv.DictReader(f):
                if tr["kernel"] == top and tr["workload"] == conf["workload"] and not bandlimit:
                    roof["traffic"] = (float(tr["dram_bytes_read"]) + float(tr["dram_bytes_write"])) * units_per_launch / float(tr["positions_per_launch"])
                    roof["traffic_source"] = tr["source"]
    except (OSError, KeyError, ValueError, StopIteration):
        pass
    # whole-step view against both roofs of SURVEY §8(d): the io+act byte model and nominal FFT flops on the FP32 ALUs
    rate = J / (ms_step * 1e-3)
    b_model = 2 * cfg.n_modes * cfg.n_slices * cfg.n * cfg.n * 8 + cfg.n * cfg.n * 4
    roof["step_model"] = {"hbm_frac_io_act_model": b_model * rate / 1e9 / hbm,
                          "fp32_frac_nominal_fft_flops": nominal_flops_per_position(cfg) * rate / 1e12 / fp32_peak,
                          "fp32_peak_tflops_at_max_clock": fp32_peak}

    # end to end through the host-buffer entry point: pinned host memory in, gradients + loss back, every step
    e2e = None
    if want_e2e:
        del ws
        torch.cuda.empty_cache()
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        obj_p, pr_p, pos_p, I_p = pin(obj_h), pin(pr_h), pin(pos_h), pin(I_h)
        gO_p = torch.empty(obj_p.shape, dtype=torch.complex64).pin_memory(); gP_p = torch.empty(pr_p.shape, dtype=torch.complex64).pin_memory()
        gX_p = torch.empty((J, 2), dtype=torch.float32).pin_memory(); loss_p = torch.zeros(1, dtype=torch.float64).pin_memory()
        wsh = ptycho.make_workspace(pbg, J, J, ptycho.WANT_POS_GRAD, host=True)

        def step_host():
            ptycho.gradient_host(pbg, obj_p, pr_p, pos_p, I_p, workspace=wsh, grad_object_h=gO_p, grad_probe_h=gP_p,
                                 grad_pos_h=gX_p, loss_h=loss_p)

        for _ in range(max(1, min(warmup, 2))):
            step_host()
        barrier()
        e0.record()
        for _ in range(steps):
            step_host()
        e1.record()
        barrier()
        msh = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device="cuda")
        if dist is not None:
            dist.all_reduce(msh, op=dist.ReduceOp.MAX)
        h2d = obj_p.numel() * 8 + pr_p.numel() * 8 + pos_p.numel() * 4 + I_p.numel() * 4
        d2h = gO_p.numel() * 8 + gP_p.numel() * 8 + gX_p.numel() * 4 + 8
        e2e = {"value": world * J / (msh.item() / steps * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h,
               "api": "ptycho_gradient_host: loss + object / probe / position gradients from and to pinned host buffers; GRADIENT ONLY - "
                      "the SGD update of `value`'s step (ptycho_apply_update, ~0.04 ms on device arrays) is not part of this loop"}
        del wsh

    cpu = None
    if rank == 0 and world == 1 and want_cpu:
        from oracle import oracle as orc
        n = args.cpu_sample or {1: 256, 2: 256, 3: 128, 4: 8, 5: 128}[cfg_idx]
        pbo = orc.Problem(**problem_kwargs(cfg))
        t0 = time.perf_counter()
        g = orc.gradient(pbo, obj_h, pr_h, pos_h, I_h, batch_idx=np.arange(n, dtype=np.int32))
        orc.apply_update(pbo, 0, obj_h, pr_h, pos_h[:n], g["grad_object"], g["grad_probe"], g["grad_pos"], **LR)
        dt = time.perf_counter() - t0
        cpu = {"value": n / dt, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
               "sample": f"first {n} of {J} positions, one forward+adjoint+update, {dt:.1f} s"}
    conf.update(parallelism=f"positions sharded over {world} GPU(s), gradients all-reduced" if world > 1 else "1 GPU",
                global_positions=world * J,
                l2_policy=(f"per-step working set {wset / 1e6:.0f} MB (patterns + stash + staging) > 126 MB L2, no flush" if flush is None else
                           f"per-step working set {wset / 1e6:.0f} MB fits L2: a 512 MB buffer is overwritten between timed steps, each "
                           "step timed with its own pair of CUDA events"),
                context=PAPER_CONTEXT)
    return dict(value=world * rate, ms_per_step=ms_step, steps=steps, warmup=warmup, config=conf, clocks=clk, e2e=e2e,
                gpu_launches=launches, roofline=roof, cpu_baseline=cpu, loss=loss_val, direct_call=direct)


TRAFFIC_FILE = "r2_dominant_kernel_traffic.csv"   # written with profiles/r2_ncu_full_summary.md
# what the default invocation times after the headline workload: (key, config, keyword overrides)
SECONDARY = [("config1", 1, {}), ("config2", 2, {}), ("config3_bandlimit_0.667", 3, dict(bandlimit=2.0 / 3.0)),
             ("config5_batch1024", 5, dict(batch=1024)), ("config4", 4, {})]


def run_b200(args):
    import torch
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1 or "RANK" in os.environ:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    common = dict(dist=dist, rank=rank, world=world, local=local)
    r = measure(args, args.config, steps=args.steps, warmup=args.warmup, bandlimit=args.bandlimit, batch=args.batch,
                want_e2e=not args.no_e2e, want_cpu=not args.no_cpu_baseline, **common)
    secondary = None
    if args.config == 3 and not args.bandlimit and not args.no_secondary and not args.stash_fp16 and world == 1:
        # the other configurations of BASELINE.json and the band-limited variant, short runs (1 warm-up + >= 2 timed steps,
        # at least one second of timed region each), device-resident only
        secondary = {}
        for key, idx, over in SECONDARY:
            torch.cuda.empty_cache()
            s = measure(args, idx, steps=2, warmup=1, want_e2e=idx in (1, 2), want_cpu=False, min_seconds=1.0, want_sweep=False,
                        prof_steps=2, **common, **over)
            rf = s["roofline"]
            secondary[key] = {"value": s["value"], "unit": UNIT, "ms_per_step": s["ms_per_step"], "steps": s["steps"], "warmup": s["warmup"],
                              "e2e": None if s["e2e"] is None else s["e2e"]["value"], "gpu_launches_per_step": s["gpu_launches"] / s["steps"],
                              "direct_call": s["direct_call"], "dominant_kernel": rf["kernel"], "frac": rf["frac"], "frac_of_measured_peak": rf.get("frac_of_measured_peak"),
                              "fp32_frac_whole_step": rf["step_model"]["fp32_frac_nominal_fft_flops"],
                              "kernel_ms_per_step": rf["kernel_ms_per_step"], "clocks": s["clocks"],
                              "workload": s["config"]["workload"], "minibatch": s["config"].get("minibatch"),
                              "variant": s["config"].get("variant"), "launch": s["config"].get("launch")}
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": r["steps"], "warmup": r["warmup"],
            "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32 (complex64)",
            "data": "synthetic", "config": r["config"], "clocks": r["clocks"], "e2e": r["e2e"], "gpu_launches": r["gpu_launches"],
            "roofline": r["roofline"], "cpu_baseline": r["cpu_baseline"], "loss": r["loss"], "direct_call": r["direct_call"], "secondary": secondary}))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_b200(a)
