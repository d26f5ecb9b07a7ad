#!/usr/bin/env python
"""bench.py — one JSON line for the RotateAttention hot path on B200.

A "step" is one pass of the whole INT4 hot path over BASELINE.json configs[1] (Wan-1.3B-like 480p:
B=1, H=12, N=32760, D=128): rotattn_prepare_qk (3D RoPE + Half rotation + INT4 Q/K) -> rotattn_quant_v ->
rotattn_fwd_int4, all through the C-ABI.  `value` = effective TOPS = 4*B*H*N^2*D / step time with inputs
resident in HBM; `e2e` = the same with HOST (pinned) Q,K,V copied in and O copied out inside the timed region.
The FP16 fallback kernel is timed beside it (speed-up denominator) but is not part of the step.
N > 1 (torchrun): every rank runs the full workload on its own GPU (independent (b,h) units, no collective);
value = total ops of all ranks / max-over-ranks time ("weak").
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = 'INT4 attn fwd effective TOPS (4*B*H*N^2*D ops per call; N=32760,H=12,D=128); ms/call in ms_per_step'
WORKLOAD = 'wan1.3b-480p'


def _peaks():
    path = os.path.join(ROOT, 'MEASURED_PEAKS.json')
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm=d['hbm_gbs'], bf16=d['bf16_tflops'], bf16_sus=d.get('bf16_tflops_sustained', d['bf16_tflops']),
                    src='MEASURED_PEAKS.json')
    return dict(hbm=6650.0, bf16=1590.0, bf16_sus=1400.0, src='fallback (B200_PROFILING.md)')


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region."""
    Q = 'clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,' \
        'clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap'

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(['nvidia-smi', '-i', str(self.index), f'--query-gpu={self.Q}',
                                          '--format=csv,noheader,nounits', '-lms', '20'],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(',')])

    def stop(self):
        if not self.proc:
            return {'sm_mhz': None, 'sm_max_mhz': None, 'reasons': ['nvidia-smi unavailable']}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace('.', '').isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace('.', '').isdigit()]
        names = ['hw_slowdown', 'hw_thermal_slowdown', 'sw_thermal_slowdown', 'sw_power_cap']
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 6 and r[2 + i].lower().startswith('active') for r in self.rows)]
        return {'sm_mhz': float(np.median(sm)) if sm else None, 'sm_max_mhz': max(mx) if mx else None, 'reasons': reasons,
                'samples': len(sm)}


def cpu_oracle_sample(n_rows=1024, threads=None):
    """Time the oracle as it stands on a bounded sample of the workload: one head's full prologue
    (RoPE + Half rotation + INT4 Q/K, V quantiser on all N tokens) + quantised attention for n_rows query rows
    against all N keys.  Returns (seconds, ops) with ops = 4*rows*N*D."""
    from oracle import rotattn_oracle as orc
    from synth import video_qkv as syn
    w = syn.ALL[WORKLOAD]
    q, k, v = syn.gen_head(w, 0, 0)
    p = orc.Params(1, 1, w.N, w.D, w.grid, w.pairs, rot_mode=orc.ROT_HALF)
    rows = syn.sample_rows(w, n_tiles=n_rows // 128, head=0)
    t0 = time.perf_counter()
    orc.int4_attention_head(p, q, k, v, rows=rows)
    dt = time.perf_counter() - t0
    return dt, 4.0 * len(rows) * w.N * w.D, len(rows)


def _time_ms(torch, fn, iters, warm=1):
    for _ in range(warm):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(iters):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / iters


def quality_report(api, syn, torch, w, Q, K, V, b, coef):
    """Quality of the INT4 path against exact attention, next to the naive symmetric-INT4 / no-rotation baseline
    (north_star).  The exact reference here is the library's own FP16 kernel on the same inputs (within 2e-3 of fp64
    attention, tests/test_gpu_fwd_fp16.py); everything runs on the GPU, heads 0..3 of the bench workload."""
    def metrics(o, ref):
        o, ref = o.double().flatten(), ref.double().flatten()
        return {'cosine': float((o @ ref) / (o.norm() * ref.norm())), 'rel_l1': float((o - ref).abs().sum() / ref.abs().sum())}
    H4 = min(4, w.H)
    out = {}
    sl = lambda t: t[:, :H4].contiguous()
    Qh, Kh, Vh = sl(Q), sl(K), sl(V)
    ref = None
    for name, rot, pm in (('half_asym15', api.ROT_HALF, api.P_ASYM15), ('interleaved_asym15', api.ROT_INTERLEAVED, api.P_ASYM15),
                          ('none_asym15', api.ROT_NONE, api.P_ASYM15), ('naive_none_sym7', api.ROT_NONE, api.P_SYM7)):
        p = api.params_for(w, rot, pm, H=H4)
        cf = torch.from_numpy(api.rotattn_build_tables(p)).cuda()
        bb = api.Buffers(p, want_fp16=ref is None)
        api.rotattn_prepare_qk(p, cf, None, Qh, Kh, bb.Q4, bb.Qs, bb.K4, bb.Ks, bb.Q16, bb.K16, bb.ws)
        api.rotattn_quant_v(p, Vh, bb.V4, bb.Vs, bb.ws)
        api.rotattn_fwd_int4(p, bb.Q4, bb.Qs, bb.K4, bb.Ks, bb.V4, bb.Vs, bb.O, bb.ws, api.WS_HAS_QK | api.WS_HAS_V)
        if ref is None:
            api.rotattn_fwd_fp16(p, bb.Q16, bb.K16, Vh, bb.O16, bb.ws16)
            ref = bb.O16.clone()
        torch.cuda.synchronize()
        out[name] = metrics(bb.O, ref)
    out['note'] = 'synthetic outlier inputs (stand-ins for Wan2.2 activations); paper reports video-level metrics only (Table 1)'
    return out


def sweep_report(api, syn, torch):
    """BASELINE.json configs[4]: H=24, D=128, N in {4096..131072}; per-N kernel ms / TOPS and the blended per-step time of
    a 50-step schedule with the FP16 fallback on the first 5 steps and on round(0.1 H) seeded heads."""
    rows = []
    for w in syn.SWEEP:
        p = api.params_for(w, api.ROT_HALF)
        B, H, N, D = w.B, w.H, w.N, w.D
        g = torch.Generator(device='cuda').manual_seed(w.seed)
        Q, K, V = (torch.randn((B, H, N, D), device='cuda', dtype=torch.float16, generator=g) for _ in range(3))
        cf = torch.from_numpy(api.rotattn_build_tables(p)).cuda()
        bb = api.Buffers(p, want_fp16=True)
        rng = np.random.Generator(np.random.PCG64(w.seed + 2))
        f16_heads = np.sort(rng.choice(H, size=max(1, round(0.1 * H)), replace=False)).astype(np.int32)
        i4_heads = np.array([h for h in range(H) if h not in set(f16_heads.tolist())], dtype=np.int32)
        sel16, sel4 = torch.from_numpy(f16_heads).cuda(), torch.from_numpy(i4_heads).cuda()
        it = 3 if N >= 65536 else 10
        ws_state = api.WS_HAS_QK | api.WS_HAS_V
        t_prep = _time_ms(torch, lambda: api.rotattn_prepare_qk(p, cf, None, Q, K, bb.Q4, bb.Qs, bb.K4, bb.Ks, bb.Q16, bb.K16, bb.ws), it)
        t_qv = _time_ms(torch, lambda: api.rotattn_quant_v(p, V, bb.V4, bb.Vs, bb.ws), it)
        t_i4 = _time_ms(torch, lambda: api.rotattn_fwd_int4(p, bb.Q4, bb.Qs, bb.K4, bb.Ks, bb.V4, bb.Vs, bb.O, bb.ws, ws_state), it)
        t_f16 = _time_ms(torch, lambda: api.rotattn_fwd_fp16(p, bb.Q16, bb.K16, V, bb.O16, bb.ws16), it)
        t_i4s = _time_ms(torch, lambda: api.rotattn_fwd_int4(p, bb.Q4, bb.Qs, bb.K4, bb.Ks, bb.V4, bb.Vs, bb.O, bb.ws, ws_state, head_sel=sel4), it)
        t_f16s = _time_ms(torch, lambda: api.rotattn_fwd_fp16(p, bb.Q16, bb.K16, V, bb.O, bb.ws16, head_sel=sel16), it)
        ops = 4.0 * B * H * N * N * D
        blended = (5 * (t_prep + t_f16) + 45 * (t_prep + t_qv + t_i4s + t_f16s)) / 50
        rows.append({'N': N, 'prepare_qk_ms': t_prep, 'quant_v_ms': t_qv, 'fwd_int4_ms': t_i4, 'fwd_int4_tops': ops / t_i4 / 1e9,
                     'fwd_fp16_ms': t_f16, 'fwd_fp16_tflops': ops / t_f16 / 1e9, 'int4_heads': len(i4_heads), 'fp16_heads': len(f16_heads),
                     'fwd_int4_subset_ms': t_i4s, 'fwd_fp16_subset_ms': t_f16s, 'blended_step_ms': blended, 'all_fp16_step_ms': t_prep + t_f16})
        del Q, K, V, bb
        torch.cuda.empty_cache()
    return rows


def run_reference(args):
    rank = int(os.environ.get('RANK', '0'))
    if rank != 0:
        return
    steps, warm = args.steps, args.warmup
    for _ in range(min(warm, 1)):
        cpu_oracle_sample(256)
    ts, ops, nrows = [], 0.0, 0
    for _ in range(max(1, min(steps, 3))):
        dt, ops, nrows = cpu_oracle_sample(2048)
        ts.append(dt)
    dt = float(np.mean(ts))
    val = ops / dt / 1e12
    sample = f'{WORKLOAD}: 1 head, full prologue on N=32760 tokens + O-quant for {nrows} query rows x all keys'
    out = {'impl': 'reference', 'metric': METRIC, 'value': val, 'unit': 'TOPS', 'n_gpus': args.gpus, 'steps': len(ts),
           'warmup': min(warm, 1), 'ms_per_step': dt * 1e3, 'higher_is_better': True, 'scaling': 'weak', 'vs_baseline': None,
           'dtype': 'f64', 'data': 'synthetic', 'config': {'workload': WORKLOAD, 'note': 'bounded sample per step: ' + sample},
           'cpu_baseline': {'value': val, 'unit': 'TOPS', 'cores': os.cpu_count(), 'kind': 'oracle', 'sample': sample},
           'e2e': {'value': val, 'unit': 'TOPS', 'h2d_bytes_per_step': 0, 'd2h_bytes_per_step': 0}, 'gpu_launches': 0}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument('--gpus', type=int, default=1)
    ap.add_argument('--steps', type=int, default=10)
    ap.add_argument('--warmup', type=int, default=3)
    ap.add_argument('--impl', default='ours')
    ap.add_argument('--no-cpu-baseline', action='store_true')
    ap.add_argument('--no-extras', action='store_true', help='skip the quality report and the N sweep (configs[4])')
    args = ap.parse_args()
    if args.impl == 'reference':
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import __graft_entry__ as entry
    entry.build()
    from paper_2607_02584_b200 import api
    from synth import video_qkv as syn

    world = int(os.environ.get('WORLD_SIZE', '1'))
    rank = int(os.environ.get('RANK', '0'))
    local = int(os.environ.get('LOCAL_RANK', '0'))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group('nccl', device_id=torch.device('cuda', local))
    W = max(3, args.warmup)
    K = args.steps
    w = syn.ALL[WORKLOAD]
    p = api.params_for(w, api.ROT_HALF)
    B, H, N, D = w.B, w.H, w.N, w.D
    ops = 4.0 * B * H * N * N * D

    # synthetic inputs of the BASELINE.json recipe (every replica runs the same seeded tensors)
    q, k, v = syn.gen_all(w)
    hq, hk, hv = (torch.from_numpy(x).pin_memory() for x in (q, k, v))
    Q, Kt, V = hq.cuda(), hk.cuda(), hv.cuda()
    coef = torch.from_numpy(api.rotattn_build_tables(p)).cuda()
    b = api.Buffers(p, want_fp16=True)
    hO = torch.empty((B, H, N, D), dtype=torch.float16).pin_memory()
    stream = torch.cuda.current_stream()

    def step():
        api.rotattn_prepare_qk(p, coef, None, Q, Kt, b.Q4, b.Qs, b.K4, b.Ks, None, None, b.ws)
        api.rotattn_quant_v(p, V, b.V4, b.Vs, b.ws)
        api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, b.O, b.ws, api.WS_HAS_QK | api.WS_HAS_V)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(ms):
        if world > 1:
            t = torch.tensor([ms], device='cuda')
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        return ms

    for _ in range(W):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    # ---- timed region: K steps, per-kernel CUDA events on the launching stream
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for i in range(K):
        ev[i][0].record(stream)
        api.rotattn_prepare_qk(p, coef, None, Q, Kt, b.Q4, b.Qs, b.K4, b.Ks, None, None, b.ws)
        ev[i][1].record(stream)
        api.rotattn_quant_v(p, V, b.V4, b.Vs, b.ws)
        ev[i][2].record(stream)
        api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, b.O, b.ws, api.WS_HAS_QK | api.WS_HAS_V)
        ev[i][3].record(stream)
    e1.record(stream)
    barrier()
    total_ms = max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop() if rank == 0 else None
    t_prep = float(np.mean([ev[i][0].elapsed_time(ev[i][1]) for i in range(K)]))
    t_qv = float(np.mean([ev[i][1].elapsed_time(ev[i][2]) for i in range(K)]))
    t_int4 = float(np.mean([ev[i][2].elapsed_time(ev[i][3]) for i in range(K)]))
    ms_step = total_ms / K

    # ---- FP16 fallback kernel (speed-up denominator), same shapes
    api.rotattn_prepare_qk(p, coef, None, Q, Kt, b.Q4, b.Qs, b.K4, b.Ks, b.Q16, b.K16, b.ws)
    for _ in range(2):
        api.rotattn_fwd_fp16(p, b.Q16, b.K16, V, b.O16, b.ws16)
    torch.cuda.synchronize()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    nf = max(2, min(K, 5))
    f0.record(stream)
    for _ in range(nf):
        api.rotattn_fwd_fp16(p, b.Q16, b.K16, V, b.O16, b.ws16)
    f1.record(stream)
    torch.cuda.synchronize()
    t_fp16 = f0.elapsed_time(f1) / nf

    # ---- end to end: host (pinned) inputs in, O out, EVERY step.  Three streams (H2D, compute, D2H) over double-buffered
    # device tensors: step i+1's inputs are copied in and step i-1's result is copied out while step i computes.
    s_in, s_c, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    Qd, Kd, Vd, Od = [Q, torch.empty_like(Q)], [Kt, torch.empty_like(Kt)], [V, torch.empty_like(V)], [b.O, torch.empty_like(b.O)]
    ev_in = [torch.cuda.Event() for _ in range(2)]
    ev_c = [torch.cuda.Event() for _ in range(2)]
    ev_out = [torch.cuda.Event() for _ in range(2)]
    ws_state = api.WS_HAS_QK | api.WS_HAS_V

    def e2e_run(n):
        for i in range(n):
            k = i & 1
            with torch.cuda.stream(s_in):
                s_in.wait_event(ev_c[k])                      # the step that last read these input buffers is done
                Qd[k].copy_(hq, non_blocking=True); Kd[k].copy_(hk, non_blocking=True); Vd[k].copy_(hv, non_blocking=True)
                ev_in[k].record(s_in)
            with torch.cuda.stream(s_c):
                s_c.wait_event(ev_in[k])
                s_c.wait_event(ev_out[k])                     # the result buffer has been copied out
                api.rotattn_prepare_qk(p, coef, None, Qd[k], Kd[k], b.Q4, b.Qs, b.K4, b.Ks, None, None, b.ws, stream=s_c)
                api.rotattn_quant_v(p, Vd[k], b.V4, b.Vs, b.ws, stream=s_c)
                api.rotattn_fwd_int4(p, b.Q4, b.Qs, b.K4, b.Ks, b.V4, b.Vs, Od[k], b.ws, ws_state, stream=s_c)
                ev_c[k].record(s_c)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_c[k])
                hO.copy_(Od[k], non_blocking=True)
                ev_out[k].record(s_out)
    e2e_run(2)
    barrier()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ne = max(4, min(K, 10))
    g0.record(s_in)
    e2e_run(ne)
    s_out.wait_stream(s_c); s_out.wait_stream(s_in)
    g1.record(s_out)
    barrier()
    e2e_ms = max_over_ranks(g0.elapsed_time(g1)) / ne
    h2d = 3 * B * H * N * D * 2
    d2h = B * H * N * D * 2

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    pk = _peaks()
    quality = sweep = None
    if not args.no_extras and world == 1:
        quality = quality_report(api, syn, torch, w, Q, Kt, V, b, coef)
        del hq, hk, hv, hO
        sweep = sweep_report(api, syn, torch)
    int8_peak = 2.0 * pk['bf16']      # dense int8 = 2x bf16 nominal ratio (4.5 / 2.25 PFLOP/s) applied to the measured bf16 peak
    achieved = ops / (t_int4 * 1e-3) / 1e12
    traffic = None
    tpath = os.path.join(ROOT, 'profiles', 'fwd_int4_traffic.csv')     # dram__bytes_read+write of one ncu --set full capture
    if os.path.exists(tpath):
        last = open(tpath).read().strip().splitlines()[-1].split(',')
        traffic = int(last[-2]) if last[-2].isdigit() else None
    out = {
        'metric': METRIC, 'value': world * ops / (ms_step * 1e-3) / 1e12, 'unit': 'TOPS', 'n_gpus': world, 'steps': K, 'warmup': W,
        'ms_per_step': ms_step, 'higher_is_better': True, 'scaling': 'weak', 'vs_baseline': None, 'dtype': 'int8 codes (INT4 values) / int32 accumulate / fp32 softmax',
        'data': 'synthetic',
        'config': {'workload': WORKLOAD, 'B': B, 'H': H, 'N': N, 'D': D, 'grid': list(w.grid), 'rot_mode': 'HALF', 'p_mode': 'ASYM15',
                   'p_norm': 'ROWBLOCK', 'l2': 'inputs larger than L2 (Q,K,V fp16 = 302 MB per step; no flush)',
                   'parallelism': f'replicas x{world} (independent (b,h) units, no collective)'},
        'kernels_ms': {'prepare_qk': t_prep, 'quant_v': t_qv, 'fwd_int4': t_int4, 'fwd_fp16': t_fp16},
        'int4_kernel_tops': achieved, 'fp16_kernel_tflops': ops / (t_fp16 * 1e-3) / 1e12,
        'speedup_int4_vs_own_fp16_kernel': t_fp16 / t_int4,
        'prologue_gbs': {'prepare_qk': (2 * (2 * D + D // 2 + 4 + 128) * B * H * N) / (t_prep * 1e-3) / 1e9,
                         'quant_v': ((2 * D + D // 2 + D) * B * H * N + 4 * D * B * H * ((N + 127) // 128)) / (t_qv * 1e-3) / 1e9,
                         'peak': pk['hbm']},
        'roofline': {'kernel': 'fwd_int4_kernel', 'bound': 'tensor', 'achieved': achieved, 'peak': int8_peak, 'unit': 'TOPS',
                     'frac': achieved / int8_peak, 'traffic': traffic,
                     'peak_source': f"2 x bf16_tflops ({pk['bf16']}) of {pk['src']} (dense int8:bf16 nominal ratio 2; of measured)"},
        'e2e': {'value': world * ops / (e2e_ms * 1e-3) / 1e12, 'unit': 'TOPS', 'ms_per_step': e2e_ms, 'how': 'C-ABI calls on pinned-host inputs; H2D / compute / D2H streams over double-buffered device tensors, every step copies all inputs in and O out',
                'h2d_bytes_per_step': h2d, 'd2h_bytes_per_step': d2h},
        'gpu_launches': 3 * K,
        'clocks': clocks,
        'paper_context': 'paper: up to 2.2x INT4 vs its FP16 kernel on A10, 1.68x end to end (PAPER.md:L267) - other hardware',
    }
    if quality is not None:
        out['quality_vs_own_fp16_kernel'] = quality
    if sweep is not None:
        out['sweep_mixed_precision'] = sweep
    if not args.no_cpu_baseline and world == 1:
        dt, cops, nrows = cpu_oracle_sample(16384)
        out['cpu_baseline'] = {'value': cops / dt / 1e12, 'unit': 'TOPS', 'cores': os.cpu_count(), 'kind': 'oracle', 'seconds': dt,
                               'sample': f'{WORKLOAD}: 1 head, full prologue on N={N} tokens + O-quant for {nrows} query rows x all keys'}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == '__main__':
    main()
