"""bench.py -- one "step" = one GW self-energy evaluation (all hot-path steps a1..a6 of DESIGN.md) on a
seeded synthetic crystal, through the C-ABI library (paper_2405_09494_b200/libgwsig.so).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--mode ibz_block] [--impl reference]

Prints ONE JSON line (rank 0).  Metric (BASELINE.json): ms per GW Sigma evaluation, plus FP64 GFLOP/s
(full-BZ-equivalent and executed) and the fraction of the FP64 tensor peak.  The default workload is
BASELINE.json configs[2] (diamond Fd-3m 6x6x6, "config 3" in the north star's 1-based count), the
largest config whose V for all wedge pairs is resident on one GPU and whose step ends in seconds;
configs[0..1] are launch-bound parity cases, configs[3..4] run with --workload cfg4 / cfg5.

Multi-GPU: the north star fixes one GPU, no sharding, no collective: "replicas
only" -- under torchrun every rank runs the same evaluation on its own GPU; the only torch.distributed
traffic is the barrier and the max-over-ranks of the device time.

--impl reference times the CPU oracle (oracle/sigma_oracle.py, as it stands) on a bounded sample of the
same workload; see DESIGN.md section 8.
"""
from __future__ import annotations

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

METRIC = "ms_per_gw_sigma_evaluation"
FP64_TENSOR_PEAK_TFLOPS = 37.2    # 148 SM x 64 FP64 FMA/clk/SM x 2 x 1.965 GHz; DMMA probe: 36.9
MODES = {"full_bz": 0, "ibz": 1, "ibz_block": 2}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="gwsig", choices=["gwsig", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--mode", default="ibz_block", choices=list(MODES))
    ap.add_argument("--no-modes", action="store_true", help="skip the FULL_BZ / IBZ comparison legs")
    ap.add_argument("--no-p0", action="store_true", help="skip the bare-bubble (Eq. 20) leg")
    ap.add_argument("--no-cfg4", action="store_true", help="default workload only: skip the cfg4 sub-record (1 warm-up + 1 step, ~3 min)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--cpu-sample-tau", type=int, default=4, help="tau points of the oracle sample")
    ap.add_argument("--ibz-nq", type=int, default=0, help="q slices timed in the IBZ comparison leg (0: all; 16 at cfg4/cfg5), scaled")
    ap.add_argument("--full-nq", type=int, default=0, help="q slices timed in the FULL_BZ comparison leg (0: 8; 2 at cfg4/cfg5), scaled")
    ap.add_argument("--engine", type=int, default=0, choices=[0, 2, 3], help="0: per-stage choice (default), 2: DMMA 4M kernel, 3: DMMA 3M kernel")
    ap.add_argument("--scratch-mib", type=int, default=0, help="main leg only: cap of the X + Y scratch in MiB (0: library default, 8192); small values "
                    "give chunks that stay in L2 at the price of many short launches (experiments)")
    ap.add_argument("--prestep", default="library", choices=["library", "torch"],
                    help="IBZ_BLOCK preparation of V (Eq. 27 transform, allowed-block detection, packing): the library's own calls "
                         "gwsig_block_maxabs / gwsig_block_transform_v (default) or the torch pre-step of presetup_device.py")
    ap.add_argument("--probe-only", action="store_true", help="print the FP64 issue-rate probes and exit")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------
# clocks (profiling recipe: sample nvidia-smi DURING the timed region)
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw = [], [], []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        seen = set()
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    seen.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(seen), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------
# workload: seeded synthetic inputs (gwsig_synth) laid out for one mode of the library
# ------------------------------------------------------------------------------------------------
class DeviceV:
    """INPUT GENERATION (not the hot path): the generator's Bloch sum (gwsig_synth.tensors.SymmetricInputs.V2_rows),
    V^{k2,k1}_{Q,bj} = sum_{R1,R2} e^{-2 pi i k2.R1 + 2 pi i k1.R2} V_{Q,b,j}(R1,R2), for lists of (k2, k1) pairs, done with
    torch on the device because a step needs thousands of pairs (and at config 5 they cannot all be resident: the compact
    real-space table is, 15 GB).  Two real GEMMs against the REAL table.  Pinned to the numpy generator by check()."""

    def __init__(self, inp, torch, dev):
        self.inp, self.torch, self.dev = inp, torch, dev
        self.Vd = torch.from_numpy(inp.Vd.reshape(len(inp.vR1) * len(inp.vR2), -1)).to(dev)      # real [nR1 nR2, nel]
        self.nel = self.Vd.shape[1]

    def dense(self, k2s, k1s):
        torch, inp = self.torch, self.inp
        fr = inp.kmesh.frac
        a2, a1 = np.asarray(k2s), np.asarray(k1s)
        f1 = np.exp(-2j * np.pi * (fr[a2] @ inp.vR1.T))              # [n, nR1]
        f2 = np.exp(+2j * np.pi * (fr[a1] @ inp.vR2.T))              # [n, nR2]
        F = (f1[:, :, None] * f2[:, None, :]).reshape(len(a1), -1)
        Fr, Fi = torch.from_numpy(np.ascontiguousarray(F.real)).to(self.dev), torch.from_numpy(np.ascontiguousarray(F.imag)).to(self.dev)
        return torch.complex(Fr @ self.Vd, Fi @ self.Vd)               # [n, naux*nao*nao]

    def check(self, k2s, k1s, V):
        for p in sorted({0, len(k1s) // 2, len(k1s) - 1}):
            ref = self.inp.V2_rows(int(k1s[p]), [int(k2s[p])])[0].ravel()
            got = V[p].reshape(-1).cpu().numpy()
            assert np.abs(got - ref).max() <= 1e-12 * max(np.abs(ref).max(), 1e-300), "device V synthesis disagrees with the generator"


class Workload:
    """inputs of one (config, mode) in the library's layout.  G, W: host arrays (device tensor for the parts that are
    only ever zero).  V: resident on the device when it fits (packed blocks in IBZ_BLOCK mode, Eq. 27 done by
    presetup_device on the GPU), else synthesised per batch of whole q into one device slot inside the step ("V is copied
    on demand": here it is re-derived on demand from the compact real-space table)."""

    def __init__(self, name, mode, B, pack, inp=None, nq_subset=None, torch=None, dev=None, device_index=0, host_only=False,
                 resident_limit_gb=110.0, q_per_batch=None, dv=None, prestep="library"):
        from gwsig_synth import make_inputs
        self.name, self.mode, self.torch, self.dev = name, mode, torch, dev
        self.dv = dv                  # the device copy of the real-space V table is shared by the legs of a run (93 GiB at cfg5)
        self.lib_prestep = prestep == "library" and mode == B.IBZ_BLOCK and torch is not None and name != "cfg1" and not host_only
        self.inp = inp if inp is not None else make_inputs(name)
        inp = self.inp
        self.lib = B.Gwsig(device=-1 if host_only else device_index)
        nq_ = None
        if name == "cfg1":
            self.cfg = pack.Configured(self.lib, mode, np.eye(3), inp.kmesh.N, inp.nao, inp.naux, inp.ntau, inp.beta, None, None, None)
            Gf, Wf = inp.G_full(), inp.W_full()
            G_of, W_of = (lambda k: Gf[k]), (lambda q: Wf[q])
        elif mode == B.FULL_BZ:
            cr = inp.cr
            self.cfg = pack.Configured(self.lib, mode, cr.a, cr.mesh, cr.nao, cr.naux, cr.ntau, cr.beta, None, None, None)
            nq_ = cr.kmesh.nk if nq_subset is None else nq_subset          # W(q) of q slices that are never pushed is never read
            G_of, W_of = inp.G_k, (lambda q: inp.W_full([q])[0])
        else:
            # the library's Eq. 27 calls need the adapted bases U handed to set_blocks (gauge S5 is recognised: no unfold is planned)
            self.cfg = pack.configure_from_crystal(self.lib, inp.cr, mode, pass_U=self.lib_prestep)
            G_of, W_of = inp.G_k, (lambda q: inp.W_full([q])[0])
        cfg = self.cfg
        if nq_ is not None and nq_ < cfg.nk:
            # FULL_BZ on a q subset: only W(q < nq) is ever read; the rest of the [Nk] buffer stays zero on the device (100 GB at cfg5)
            self.G = np.ascontiguousarray(np.stack([G_of(int(k)) for k in range(cfg.nk)]).ravel(), np.complex128)
            # the library reads W(q) only for the q it is given pairs of: the buffer holds the first nq slices (100 GB in full at cfg5)
            self.W = np.ascontiguousarray(np.stack([W_of(int(q)) for q in range(nq_)]).ravel(), np.complex128)
        else:
            self.G, self.W = cfg.pack_GW(G_of, W_of)
        self.nq = cfg.nk if nq_subset is None else min(nq_subset, cfg.nk)      # q slices actually pushed
        self.npairs_run = self.nq * cfg.nk1
        self.resident = True
        self.setup_notes = {}
        if name == "cfg1" or torch is None:
            self.V = cfg.pack_V(inp.V2_rows)
        else:
            self._device_V(B, resident_limit_gb, q_per_batch)
        self.full_equiv, self.executed = self.lib.flop_counts()
        self.executed_run = self.executed * self.nq / cfg.nk if self.nq != cfg.nk else self.executed

    # ---- V on the device ---------------------------------------------------------------------------------
    def _pairs(self, p0, p1):
        cfg = self.cfg
        k1s = [int(cfg.out_list[p % cfg.nk1]) for p in range(p0, p1)]
        qs = [p // cfg.nk1 for p in range(p0, p1)]
        k2s = [int(self.inp.kmesh.sub(k1, q)) for k1, q in zip(k1s, qs)]
        return qs, k2s, k1s

    def _device_V(self, B, resident_limit_gb, q_per_batch):
        torch, dev, cfg, lib = self.torch, self.dev, self.cfg, self.lib
        t0 = time.time()
        if self.dv is None:
            self.dv = DeviceV(self.inp, torch, dev)
        nel = self.dv.nel
        nk1 = cfg.nk1
        qb = q_per_batch or max(1, int(2.0e9 // (nk1 * nel * 16)))            # ~2 GB of dense V per generation batch
        self.batches = [(q0 * nk1, min(q0 + qb, self.nq) * nk1) for q0 in range(0, self.nq, qb)]
        blockmode = self.mode == B.IBZ_BLOCK
        if blockmode:
            if not self.lib_prestep:
                from paper_2405_09494_b200.presetup_device import DeviceBlocker
                self.blk = DeviceBlocker(cfg, torch, dev)
            else:
                mb_aux = max(len(o) - 1 for o in cfg.aux.off)
                mb_ao = max(len(o) - 1 for o in cfg.ao.off)
            # pass 1 (pre-step, all pairs of the mode: set_triples wants every pair): allowed blocks by block max-abs
            trip, vmax = [], None
            allb = [(q0 * nk1, min(q0 + qb, cfg.nk) * nk1) for q0 in range(0, cfg.nk, qb)]
            for bi, (p0, p1) in enumerate(allb):
                qs, k2s, k1s = self._pairs(p0, p1)
                V = self.dv.dense(k2s, k1s)
                if bi == 0:
                    self.dv.check(k2s, k1s, V)
                    vmax = float(V.abs().max())
                if self.lib_prestep:
                    # Eq. 27 for every block + block maxima in the library (gwsig_block_maxabs), thresholded here
                    dM = torch.empty((p1 - p0, mb_aux, mb_ao, mb_ao), dtype=torch.float64, device=dev)
                    lib.block_maxabs(p0, p1 - p0, V.contiguous(), mb_aux, mb_ao, dM, torch.cuda.current_stream().cuda_stream)
                    mx = dM.cpu().numpy()
                    trip += [np.argwhere(m > 1e-9 * vmax).astype(np.int32) for m in mx]
                    del V, dM
                else:
                    T = self.blk.transform(V.reshape(len(k1s), cfg.naux, cfg.nao, cfg.nao), qs, k2s, k1s)
                    del V
                    trip += self.blk.triples_from_maxabs(self.blk.block_maxabs(T, qs, k2s, k1s), qs, k2s, k1s, 1e-9, vmax)
                    del T
            tptr = np.zeros(cfg.npairs + 1, np.int64)
            tptr[1:] = np.cumsum([len(t) for t in trip])
            lib.set_triples(tptr, np.concatenate(trip))
            cfg.triple_ptr, cfg.triples = tptr, trip
            if self.lib_prestep:
                self.voff = np.array([lib.pair_info(p)[3] for p in range(self.npairs_run)] + [0], np.int64)
                last = lib.pair_info(self.npairs_run - 1)
                self.voff[-1] = last[3] + last[4]
            else:
                self.tables = []
                for (p0, p1) in self.batches:
                    qs, k2s, k1s = self._pairs(p0, p1)
                    self.tables.append(self.blk.pack_tables(trip[p0:p1], qs, k2s, k1s))
                sizes = np.concatenate([t[3] for t in self.tables])
                assert all(int(sizes[i]) == lib.pair_info(i)[4] for i in (0, len(sizes) // 2, len(sizes) - 1)), "packed V layout mismatch"
                self.voff = np.concatenate([[0], np.cumsum(sizes)])
        else:
            self.voff = np.arange(self.npairs_run + 1, dtype=np.int64) * nel
        total_gb = float(self.voff[-1]) * 16 / 1e9
        self.resident = total_gb <= resident_limit_gb
        self.setup_notes = {"v_total_gb": round(total_gb, 2), "v_resident": self.resident, "q_per_generation_batch": qb}
        if self.resident:
            self.V = torch.empty(int(self.voff[-1]), dtype=torch.complex128, device=dev)
            for bi in range(len(self.batches)):
                self.fill(bi, self.V, int(self.voff[self.batches[bi][0]]), check=(bi == 0 and not blockmode))
        else:
            slot = max(int(self.voff[p1] - self.voff[p0]) for p0, p1 in self.batches)
            self.V = None
            self.slot = torch.empty(slot, dtype=torch.complex128, device=dev)
        self.setup_notes["v_setup_s"] = round(time.time() - t0, 1)

    def fill(self, bi, dst, base, check=False):
        """dense Bloch sum (+ Eq. 27 transform and packing in block mode) of generation batch bi into dst[base:]."""
        p0, p1 = self.batches[bi]
        qs, k2s, k1s = self._pairs(p0, p1)
        V = self.dv.dense(k2s, k1s)
        if check:
            self.dv.check(k2s, k1s, V)
        if self.mode == 2 and self.lib_prestep:
            # Eq. 27 on the allowed blocks, written straight into the packed layout by the library (gwsig_block_transform_v)
            self.lib.block_transform_v(p0, p1 - p0, V.contiguous(), dst[base:], self.torch.cuda.current_stream().cuda_stream)
            del V
        elif self.mode == 2:
            cfg = self.cfg
            T = self.blk.transform(V.reshape(len(k1s), cfg.naux, cfg.nao, cfg.nao), qs, k2s, k1s)
            del V
            self.blk.pack(T, qs, k2s, k1s, self.tables[bi], dst, (self.voff[p0:p1] - self.voff[p0]) + base)
        else:
            dst[base:base + V.numel()] = V.reshape(-1)

    def evaluate(self, dG, dW, dS, stream, dV=None):
        """enqueue ONE evaluation: resident V -> sigma_eval; otherwise begin / per batch {synthesise into the slot, push} / end."""
        lib, cfg = self.lib, self.cfg
        partial = self.npairs_run != cfg.npairs
        if self.resident and not partial:
            lib.sigma_eval(dG, dV, dW, dS, stream)
            return
        lib.sigma_begin(dG, dW, dS, stream)
        if self.resident:
            lib.sigma_push_pairs(0, self.npairs_run, dV)
        else:
            for bi, (p0, p1) in enumerate(self.batches):
                self.fill(bi, self.slot, 0)                       # same stream: the slot is rewritten after the previous push drained
                lib.sigma_push_pairs(p0, p1 - p0, self.slot)
        if partial:
            lib.sigma_abort()
        else:
            lib.sigma_end()


def stage_flops(wl, B):
    """algorithmic real flops of stages 1, 2, 3 of one evaluation (8 per complex MAC), from the plan's descriptors."""
    lib, cfg = wl.lib, wl.cfg
    out = []
    for stage in (1, 2, 3):
        prob, seg, _ = lib.plan_get(0, wl.npairs_run, 1, stage)
        macs = 0.0
        for P in prob:
            K = sum(int(seg[s]["K"]) for s in range(P["seg_begin"], P["seg_begin"] + P["seg_count"]))
            macs += float(P["M"]) * float(P["N"]) * K * int(P["nbatch"])
        out.append(8.0 * macs * cfg.ntau)
    return out


# ------------------------------------------------------------------------------------------------
# timed legs
# ------------------------------------------------------------------------------------------------
def to_dev(x, torch, dev):
    return x if torch.is_tensor(x) else torch.from_numpy(x).to(dev)


def run_steps(wl, torch, dev, steps, warmup, timing=True):
    """K evaluations (G, W and -- when it fits -- V resident in HBM); device time by CUDA events on the launching stream.
    Returns (seconds per step list, per-kind kernel times of the last step, launches per step, dSigma)."""
    lib = wl.lib
    dG, dW = to_dev(wl.G, torch, dev), to_dev(wl.W, torch, dev)
    dV = to_dev(wl.V, torch, dev) if wl.V is not None else None
    dS = torch.zeros(lib.buffer_sizes()[2], dtype=torch.complex128, device=dev)
    stream = torch.cuda.current_stream().cuda_stream
    lib.set_option("timing", 1 if timing else 0)
    for _ in range(warmup):
        wl.evaluate(dG, dW, dS, stream, dV)
    torch.cuda.synchronize()
    times = []
    for _ in range(steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        wl.evaluate(dG, dW, dS, stream, dV)
        e1.record()
        e1.synchronize()
        times.append(e0.elapsed_time(e1) * 1e-3)
    kinds = lib.kernel_times() if timing else {}
    return times, kinds, lib.last_launch_count(), dS


def run_e2e(wl, torch, dev, steps, warmup):
    """the same evaluation through gwsig_sigma_eval_host: inputs in PINNED HOST memory, Sigma read back to the host,
    all copies inside the timed region (wall clock around a call that returns after the result has landed)."""
    lib = wl.lib
    hG, hW = torch.from_numpy(wl.G).pin_memory(), torch.from_numpy(wl.W).pin_memory()
    hV = (wl.V.cpu() if torch.is_tensor(wl.V) else torch.from_numpy(wl.V)).pin_memory()
    hS = torch.zeros(lib.buffer_sizes()[2], dtype=torch.complex128).pin_memory()
    stream = torch.cuda.current_stream().cuda_stream
    lib.set_option("timing", 0)
    for _ in range(warmup):
        lib.sigma_eval_host(hG, hV, hW, hS, stream)
    torch.cuda.synchronize()
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        lib.sigma_eval_host(hG, hV, hW, hS, stream)
        times.append(time.perf_counter() - t0)
    h2d = (hG.numel() + hW.numel() + hV.numel()) * 16
    d2h = hS.numel() * 16
    return times, h2d, d2h, hS.numpy().copy()


def oracle_sample(inp, ks, taus):
    """the CPU oracle (oracle/sigma_oracle.py, as it stands) on a sample of (k, tau) outputs, with its inputs generated
    before the clock starts.  Returns (seconds, Sigma[len(ks), len(taus), nao, nao], threads)."""
    from oracle.sigma_oracle import sigma_ref
    taus = np.asarray(taus)
    nk = inp.nk
    Gs = {k: (inp.G_k(k) if hasattr(inp, "G_k") else inp.G_full()[k])[taus] for k in range(nk)}
    Ws = {q: inp.W_full([q])[0][taus] for q in range(nk)}
    Vs = {}
    for k in ks:
        k2s = list(range(nk))
        rows2 = inp.V2_rows(int(k), k2s)                   # V^{k2,k}
        rows1 = inp.V1_rows(int(k), k2s)                   # V^{k,k2}: generated independently, not by conjugation
        for k2 in k2s:
            Vs[(k2, int(k))] = rows2[k2]
            Vs[(int(k), k2)] = rows1[k2]
    t0 = time.perf_counter()
    out = sigma_ref(nk, inp.kmesh.sub, lambda k: Gs[k], lambda q: Ws[q], lambda a, b: Vs[(a, b)], ks)
    dt = time.perf_counter() - t0
    try:
        import threadpoolctl
        thr = max([p["num_threads"] for p in threadpoolctl.threadpool_info()] or [1])
    except Exception:
        thr = os.cpu_count() or 1
    return dt, out, thr


def fold_and_compare(wl, sigma_flat, ref, ks, taus):
    """GPU Sigma (layout of the mode) -> orbital basis at the sampled wedge points (test-side fold, Eq. 26) and the max
    relative Frobenius error per (k, tau) against the oracle sample."""
    cfg = wl.cfg
    S = cfg.unpack_sigma(sigma_flat)
    pos = {int(k): i for i, k in enumerate(cfg.out_list)}
    worst = 0.0
    for a, k in enumerate(ks):
        M = S[pos[int(k)]]
        if cfg.mode == 2:
            U = cfg.ao.U[int(k)]
            M = U @ M @ U.conj().T
        for b, t in enumerate(taus):
            worst = max(worst, float(np.linalg.norm(M[t] - ref[a, b]) / max(np.linalg.norm(ref[a, b]), 1e-300)))
    return worst


def p0_leg(inp, B, pack, torch, dev, local, engine, dv, steps=2, warmup=1, with_oracle=True):
    """N1: one bare-bubble evaluation P0^q(tau) (Eq. 20, Algorithm 3) for the wedge q of the same crystal, dense IBZ mode,
    V^{k,k+q} for all Nk x nik pairs synthesised on the device (input generation) and resident; checked against
    oracle/p0_oracle.py at one (q, tau) pair of outputs."""
    lib = B.Gwsig(device=local)
    cfg = pack.configure_from_crystal(lib, inp.cr, B.IBZ)
    lib.set_option("engine", engine)
    nk, nq = cfg.nk, len(cfg.out_list)
    zero_w = np.zeros((1, 1, 1), complex)
    G = np.ascontiguousarray(np.stack([inp.G_k(int(k)) for k in cfg.ir_list]).ravel(), np.complex128)
    km = inp.kmesh
    ks = [k for k in range(nk) for _ in range(nq)]
    kqs = [int(km.index(km.n[k] + km.n[int(q)])) for k in range(nk) for q in cfg.out_list]
    if dv is None:
        dv = DeviceV(inp, torch, dev)
    V = torch.empty((len(ks), dv.nel), dtype=torch.complex128, device=dev)
    for s0 in range(0, len(ks), 256):
        V[s0:s0 + 256] = dv.dense(ks[s0:s0 + 256], kqs[s0:s0 + 256])           # V^{k,k+q}: first momentum k, second k+q
    dG = torch.from_numpy(G).to(dev)
    dP = torch.zeros(nq * cfg.ntau * cfg.naux ** 2, dtype=torch.complex128, device=dev)
    stream = torch.cuda.current_stream().cuda_stream
    lib.set_option("timing", 1)
    for _ in range(warmup):
        lib.p0_eval(dG, V, dP, stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        lib.p0_eval(dG, V, dP, stream)
    e1.record()
    e1.synchronize()
    ms = e0.elapsed_time(e1) / steps
    kinds = lib.kernel_times()
    A_, B_ = float(cfg.naux) * cfg.nao ** 3, float(cfg.naux) ** 2 * cfg.nao ** 2
    flops = 8.0 * nk * nq * cfg.ntau * (2 * A_ + B_)
    rec = {"what": "bare bubble P0^q(tau), Eq. 20 / Algorithm 3, q in the wedge, dense blocks", "ms": ms, "pairs": nk * nq,
           "gflop_algorithmic": flops / 1e9, "tflops": flops / (ms * 1e-3) / 1e12, "frac_fp64_tensor_peak": flops / (ms * 1e-3) / 1e12 / FP64_TENSOR_PEAK_TFLOPS,
           "kernels_ms": {k: round(v[0], 2) for k, v in kinds.items() if v[1]}, "gpu_launches": int(lib.last_launch_count())}
    if with_oracle:
        from oracle.p0_oracle import p0_ref
        iq, taus = nq - 1, [0, cfg.ntau // 2]
        q = int(cfg.out_list[iq])
        kq_of = lambda k: int(km.index(km.n[k] + km.n[q]))
        Va = inp.V_pairs(list(range(nk)), [kq_of(k) for k in range(nk)])          # V^{k,k+q}
        Vb = inp.V_pairs([kq_of(k) for k in range(nk)], list(range(nk)))          # V^{k+q,k}: generated independently
        Gc = {}

        def G_of(k):
            if k not in Gc:
                Gc[k] = inp.G_k(k)
            return Gc[k]
        t0 = time.perf_counter()
        calls = {"n": 0}

        def V_pair(a, b):            # p0_ref asks for V^{k,k+q} (first momentum k = a) first, then V^{k+q,k} (second momentum k = b)
            calls["n"] += 1
            return Va[a] if calls["n"] % 2 == 1 else Vb[b]
        ref = p0_ref(nk, lambda k, q_: kq_of(k), G_of, V_pair, [q], taus)[0]
        got = dP.cpu().numpy().reshape(nq, cfg.ntau, cfg.naux, cfg.naux)[iq][taus]
        rec["parity_sample_max_rel_err"] = float(max(np.linalg.norm(got[i] - ref[i]) / np.linalg.norm(ref[i]) for i in range(len(taus))))
        rec["parity_sample"] = f"q={q}, tau idx={taus}, oracle {time.perf_counter() - t0:.1f} s"
    return rec


def sample_points(cfg_ir_list, ntau, nk_sample, ntau_sample):
    ks = [int(cfg_ir_list[0]), int(cfg_ir_list[-1])][:nk_sample] if len(cfg_ir_list) > 1 else [int(cfg_ir_list[0])]
    taus = sorted(set(np.linspace(0, ntau - 1, ntau_sample).round().astype(int).tolist()))
    return ks, taus


def replicas_step_time(secs_local, steps, world, dist=None, torch=None, device=None):
    """the N > 1 rule of this bench (replicas only, no data-path collective): every rank evaluates the
    same Sigma on its own GPU; the step time is the MAX over ranks of the device-timed region (one all_reduce of one double),
    and `world` evaluations finish per step, so the whole-job metric is step time / world.  Returns (ms_per_step, ms_per_evaluation)."""
    secs = float(secs_local)
    if world > 1:
        t = torch.tensor([secs], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        secs = float(t.item())
    ms_step = secs / steps * 1e3
    return ms_step, ms_step / world


def reference_main(args, rank, world):
    """--impl reference: the oracle as it stands on the host cores, on a bounded sample of the same workload."""
    if rank != 0:
        return
    from gwsig_synth import make_inputs
    inp = make_inputs(args.workload)
    if args.workload == "cfg1":
        ir = list(range(inp.nk))
    else:
        ir = [int(k) for k in inp.kmesh.stars(inp.cr.sg)[0]]       # the generator's own star finder: no product code in this arm
    ks, taus = sample_points(ir, inp.ntau, 1, args.cpu_sample_tau)
    for _ in range(max(args.warmup, 0)):
        oracle_sample(inp, ks[:1], taus[:1])
    tot, thr = 0.0, 1
    for _ in range(max(args.steps, 1)):
        dt, _, thr = oracle_sample(inp, ks, taus)
        tot += dt
    per_out = tot / max(args.steps, 1) / (len(ks) * len(taus))
    ms_full = per_out * inp.nk * inp.ntau * 1e3
    sample = (f"{len(ks)} k x {len(taus)} tau outputs of {args.workload} per step, full-BZ no-symmetry oracle; value = measured s per "
              f"(k,tau) output x Nk x ntau (extrapolated to one whole evaluation)")
    line = {"impl": "reference", "metric": METRIC, "value": ms_full, "unit": "ms", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": tot / max(args.steps, 1) * 1e3, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "complex128 (f64)", "data": "synthetic",
            "config": {"workload": args.workload, "mode": "full_bz oracle sample"},
            "cpu_baseline": {"value": ms_full, "unit": "ms", "cores": thr, "kind": "oracle", "sample": sample},
            "e2e": {"value": ms_full, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the committed `ncu --set full`
# capture of this command (profiles/r2_ncu_default_engine_cfg3.md, r2_ncu_cfg4_stages12.md); ncu never runs inside bench.py, so every other
# (workload, mode, engine) reports null.  Key: (workload, mode, engine option, stage index 0..2).
NCU_DRAM_BYTES_PER_LAUNCH = {("cfg3", "ibz_block", 0, 1): 7.72e9,
                             ("cfg4", "ibz_block", 0, 1): 11.23e9}   # cfg4: a generic-q launch (profiles/r2_ncu_cfg4_stages12.md); launch sizes vary with q


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        reference_main(args, rank, world)
        return
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    from paper_2405_09494_b200 import build as gw_build
    if rank == 0:
        gw_build.build()
    if world > 1:
        dist.barrier()
    from paper_2405_09494_b200 import binding as B, pack

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.probe_only:
        lib = B.Gwsig(device=local)
        out = {}
        for kind, nm in ((0, "dmma"), (1, "dfma"), (2, "dmma+dfma interleaved")):
            best = 0.0
            for w, bps in ((4, 2), (8, 2), (8, 4), (16, 2), (16, 4)):
                best = max(best, lib.probe_fp64(kind, w, bps, 20000)[0])
            out[nm] = best
        tf1, ms1 = lib.probe_fp64(3, 4, 1, 20000)        # one chain per warp, one warp per SM sub-partition
        n_dmma = 20000 * 16
        sm_hz = 1.965e9
        lat = {"dependent_dmma_cycles_at_1965MHz": ms1 * 1e-3 * sm_hz / n_dmma, "ms": ms1, "chain_length": n_dmma}
        print(json.dumps({"fp64_probe_tflops": out, "dmma_issue_cycles_per_subpartition": 512.0 * 148 * 4 * sm_hz / (out["dmma"] * 1e12),
                          "dmma_latency": lat}))
        return

    mode = MODES[args.mode]
    if args.workload == "cfg1":
        mode = B.FULL_BZ
    t_setup = time.time()
    wl = Workload(args.workload, mode, B, pack, torch=torch, dev=dev, device_index=local, prestep=args.prestep)
    cfg, lib = wl.cfg, wl.lib
    lib.set_option("engine", args.engine)
    if args.scratch_mib > 0:
        lib.set_option("scratch_mib", args.scratch_mib)
    t_setup = time.time() - t_setup

    # ---- the timed region: W warm-up steps, then exactly K steps between barrier + synchronize --------------
    dG, dW = to_dev(wl.G, torch, dev), to_dev(wl.W, torch, dev)
    dV = to_dev(wl.V, torch, dev) if wl.V is not None else None
    dS = torch.zeros(lib.buffer_sizes()[2], dtype=torch.complex128, device=dev)
    stream = torch.cuda.current_stream().cuda_stream
    lib.set_option("timing", 1)
    for _ in range(args.warmup):
        wl.evaluate(dG, dW, dS, stream, dV)
    barrier()
    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        wl.evaluate(dG, dW, dS, stream, dV)
    e1.record()
    barrier()
    secs = e0.elapsed_time(e1) * 1e-3
    clocks = sampler.stop()
    kinds = lib.kernel_times()
    launches = lib.last_launch_count()
    ms_step, ms_eval = replicas_step_time(secs, args.steps, world, dist, torch, dev)     # max over ranks; `world` evaluations per step
    sigma_gpu = dS.cpu().numpy()
    dV = None

    line = {"metric": METRIC, "value": ms_eval, "unit": "ms", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex128 (f64)", "data": "synthetic",
            "config": {"workload": f"{args.workload} ({describe(args.workload)})", "mode": args.mode, "engine": {0: "dmma (3M stages 1 and 2, 4M stage 3)", 2: "dmma 4M", 3: "dmma 3M"}[args.engine], "nk": int(cfg.nk), "nik": int(cfg.nk1),
                       "nao": int(cfg.nao), "naux": int(cfg.naux), "ntau": int(cfg.ntau), "pairs": int(cfg.npairs),
                       "l2": "inputs larger than L2 (V alone is %.2f GB)" % (wl.setup_notes.get("v_total_gb") or wl.V.nbytes / 1e9),
                       "v": ("resident in HBM" if wl.resident else "synthesised on the device per batch of whole q INSIDE the step (all pairs do not fit HBM): "
                             "value includes that input generation, kernels_last_step is the library alone"),
                       **wl.setup_notes,
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "setup_s": round(t_setup, 1)},
            "gpu_launches": int(launches) * args.steps, "clocks": clocks}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    sys.stderr.write("[bench] main leg: %.1f ms per evaluation, kernels %s\n" % (ms_eval, {k: round(v[0], 1) for k, v in kinds.items()}))
    sys.stderr.flush()

    # ---- accounting: flops, stage shares, roofline ------------------------------------------------------------
    sf = stage_flops(wl, B)
    t1, t2, t3 = (kinds[k][0] * 1e-3 for k in ("stage1_X=VG", "stage2_Y=WX", "stage3_S+=YV"))
    peak = FP64_TENSOR_PEAK_TFLOPS
    line["gflops_full_bz_equivalent"] = wl.full_equiv / (ms_eval * 1e-3) / 1e9
    line["gflops_executed"] = wl.executed / (ms_eval * 1e-3) / 1e9
    line["frac_fp64_tensor_peak_whole_step"] = wl.executed / (ms_eval * 1e-3) / 1e12 / peak
    line["kernels_last_step"] = {k: {"ms": round(v[0], 3), "launches": v[1]} for k, v in kinds.items()}
    line["contraction"] = {"tflops": (sf[0] + sf[1] + sf[2]) / max(t1 + t2 + t3, 1e-12) / 1e12,
                           "frac_fp64_tensor_peak": (sf[0] + sf[1] + sf[2]) / max(t1 + t2 + t3, 1e-12) / 1e12 / peak,
                           "stage_tflops": [sf[0] / max(t1, 1e-12) / 1e12, sf[1] / max(t2, 1e-12) / 1e12, sf[2] / max(t3, 1e-12) / 1e12],
                           "stage_gflop": [x / 1e9 for x in sf]}
    probe_tf = max(lib.probe_fp64(0, w, b, 20000)[0] for w, b in ((8, 2), (16, 2)))
    dom = int(np.argmax([t1, t2, t3]))
    ach = sf[dom] / max((t1, t2, t3)[dom], 1e-12) / 1e12
    line["roofline"] = {"bound": "tensor", "kernel": ("stage1_X=VG", "stage2_Y=WX", "stage3_S+=YV")[dom] + (" (zgemm_grouped_dmma3m)" if (args.engine == 3 or (args.engine == 0 and dom in (0, 1))) else " (zgemm_grouped_dmma)"),
                        "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                        "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get((args.workload, args.mode, args.engine, dom)),
                        "traffic_note": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, profiles/r2_ncu_default_engine_cfg3.md): "
                                        "X is read from and Y written to HBM; null where no ncu capture of this command is committed",
                        "peak_measured_dmma_probe": probe_tf,
                        "peak_source": "FP64 tensor (DMMA) peak derived from unit counts x max clock, 148 x 128 flop/clk x 1.965 GHz "
                                       "(MEASURED_PEAKS.json has no FP64 entry); peak_measured_dmma_probe is the register-only DMMA issue-rate "
                                       "probe of this library (gwsig_probe_fp64) run in this job",
                        "note": "achieved counts ALGORITHMIC flops (8 per complex multiply-add); the 3M kernel executes 6 per complex "
                                "multiply-add on the pipe, so a fully busy pipe would read 1.33"}

    # ---- end to end through the host-buffer call ------------------------------------------------------------------
    if not args.no_e2e and wl.resident and wl.setup_notes.get("v_total_gb", 0) <= 16:
        et, h2d, d2h, hs = run_e2e(wl, torch, dev, args.steps, max(1, min(args.warmup, 2)))
        line["e2e"] = {"value": float(np.mean(et)) * 1e3, "unit": "ms", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                       "api": "gwsig_sigma_eval_host (pinned host G, W, V -> host Sigma; V streamed through a 2-slot ring)"}
        assert np.abs(hs - sigma_gpu).max() <= 1e-12 * np.abs(sigma_gpu).max(), "host-buffer path disagrees with the resident path"

    # ---- CPU oracle beside it (baseline, and a live parity sample) ------------------------------------------------
    if not args.no_cpu_baseline:
        ir = list(range(cfg.nk)) if mode == B.FULL_BZ else list(cfg.ir_list)
        ks, taus = sample_points(ir, cfg.ntau, 2, args.cpu_sample_tau)
        dt, ref, thr = oracle_sample(wl.inp, ks, taus)
        per_out = dt / (len(ks) * len(taus))
        from oracle.sigma_oracle import flops_per_output
        line["cpu_baseline"] = {"value": per_out * cfg.nk * cfg.ntau * 1e3, "unit": "ms", "cores": thr, "kind": "oracle",
                                "sample": f"{len(ks)} k x {len(taus)} tau outputs (k={ks}, tau idx={taus}) in {dt:.1f} s; value = s per (k,tau) "
                                          f"output x Nk x ntau, extrapolated to a whole full-BZ no-symmetry evaluation",
                                "gflops": flops_per_output(cfg.nk, cfg.nao, cfg.naux) / per_out / 1e9}
        line["parity_sample_max_rel_err"] = fold_and_compare(wl, sigma_gpu, ref, ks, taus)

    # ---- speedup of symmetry adaptation: the other modes on the same crystal, all on the GPU ----------------------
    if not args.no_modes and args.workload != "cfg1":
        modes = {args.mode: {"ms": ms_eval, "gflop_executed": wl.executed / 1e9}}
        wl.V = None
        if hasattr(wl, "slot"):
            del wl.slot
        torch.cuda.empty_cache()
        big = args.workload in ("cfg4", "cfg5")
        for mname, nq in (("ibz", args.ibz_nq or (16 if big else None)), ("full_bz", args.full_nq or (2 if big else 8))):
            if mname == args.mode:
                continue
            w2 = Workload(args.workload, MODES[mname], B, pack, inp=wl.inp, nq_subset=nq, torch=torch, dev=dev, device_index=local,
                          dv=getattr(wl, "dv", None))
            w2.lib.set_option("engine", args.engine)
            tt, k2, _, _ = run_steps(w2, torch, dev, 1, 1, timing=(mname == "ibz"))
            scale = w2.cfg.nk / w2.nq
            modes[mname] = {"ms": tt[0] * 1e3 * scale, "gflop_executed": w2.executed / 1e9}
            if mname == "ibz":
                # the HBM-bound helper kernels of the IBZ mode (steps a1, a2): algorithmic bytes = unfolded output written once
                # + the wedge source read once, against the measured copy bandwidth (MEASURED_PEAKS.json hbm_gbs)
                c2 = w2.cfg
                nik = len(c2.ir_list)
                bg = 16.0 * c2.ntau * c2.nao ** 2 * (c2.nk + nik)
                bw = 16.0 * c2.ntau * c2.naux ** 2 * (w2.nq + min(nik, w2.nq))
                ug, uw = k2["unfold_G"][0] * 1e-3, k2["unfold_W"][0] * 1e-3
                hbm = measured_hbm_gbs()
                modes[mname]["unfold"] = {"G_ms": ug * 1e3, "W_ms": uw * 1e3, "G_gbs": bg / max(ug, 1e-12) / 1e9, "W_gbs": bw / max(uw, 1e-12) / 1e9,
                                          "hbm_peak_gbs": hbm, "W_frac_of_measured_hbm": bw / max(uw, 1e-12) / 1e9 / hbm,
                                          "share_of_step": (ug + uw) / tt[0]}
            if scale != 1:
                modes[mname]["note"] = f"timed on the first {w2.nq} of {w2.cfg.nk} q slices (all k1, all tau; every slice costs the same), scaled x{scale:g}"
            del w2
            torch.cuda.empty_cache()
        base = modes.get("full_bz", {}).get("ms")
        if base:
            for m in modes.values():
                m["speedup_vs_full_bz"] = base / m["ms"]
        line["modes"] = modes

    # ---- N1: the bare bubble on the same crystal -------------------------------------------------------------------------------
    if args.workload in ("cfg2", "cfg3") and not args.no_p0 and world == 1:
        wl.V = None
        torch.cuda.empty_cache()
        line["p0"] = p0_leg(wl.inp, B, pack, torch, dev, local, args.engine, getattr(wl, "dv", None), with_oracle=not args.no_cpu_baseline)

    # ---- the other target config of the north star (configs 3-4): one step of cfg4 in the same job ------------------------------
    if args.workload == "cfg3" and not args.no_cfg4 and world == 1:
        wl.V = None
        dG = dW = dS = None
        torch.cuda.empty_cache()
        t4 = time.time()
        w4 = Workload("cfg4", MODES[args.mode], B, pack, torch=torch, dev=dev, device_index=local, prestep=args.prestep)
        w4.lib.set_option("engine", args.engine)
        tt, k4, l4, dS4 = run_steps(w4, torch, dev, 1, 1, timing=True)
        sf4 = stage_flops(w4, B)
        ts4 = [k4[k][0] * 1e-3 for k in ("stage1_X=VG", "stage2_Y=WX", "stage3_S+=YV")]
        rec = {"workload": describe("cfg4"), "mode": args.mode, "steps": 1, "warmup": 1, "ms": tt[0] * 1e3,
               "gflops_executed": w4.executed / tt[0] / 1e9, "gflops_full_bz_equivalent": w4.full_equiv / tt[0] / 1e9,
               "kernels_ms": {k: round(v[0], 2) for k, v in k4.items()}, "gpu_launches": int(l4),
               "contraction": {"tflops": sum(sf4) / max(sum(ts4), 1e-12) / 1e12, "frac_fp64_tensor_peak": sum(sf4) / max(sum(ts4), 1e-12) / 1e12 / peak,
                               "stage_tflops": [f / max(t, 1e-12) / 1e12 for f, t in zip(sf4, ts4)]},
               **w4.setup_notes}
        if not args.no_cpu_baseline:
            ks4, taus4 = sample_points(list(w4.cfg.ir_list), w4.cfg.ntau, 1, 2)
            dt4, ref4, _ = oracle_sample(w4.inp, ks4, taus4)
            rec["parity_sample_max_rel_err"] = fold_and_compare(w4, dS4.cpu().numpy(), ref4, ks4, taus4)
            rec["parity_sample"] = f"k={ks4}, tau idx={taus4}, oracle {dt4:.1f} s"
        rec["wall_s"] = round(time.time() - t4, 1)
        line["cfg4"] = rec
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def measured_hbm_gbs():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        return 6650.0            # the profiling guide's fallback


def describe(name):
    return {"cfg1": "BASELINE configs[0]: C1 2x2x2, nao 8, naux 32, ntau 16",
            "cfg2": "BASELINE configs[1]: simple cubic Oh 4x4x4, nao 9, naux 18, ntau 64",
            "cfg3": "BASELINE configs[2]: diamond Fd-3m 6x6x6, nao 26, naux 116, ntau 104",
            "cfg4": "BASELINE configs[3]: wurtzite P6_3mc 6x6x4, nao 52, naux 232, ntau 128",
            "cfg5": "BASELINE configs[4]: rock salt Fm-3m 8x8x8, nao 58, naux 300, ntau 136"}[name]


if __name__ == "__main__":
    main()
