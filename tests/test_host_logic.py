"""CPU-only tests of the product's host side (no GPU): the C-ABI library loads and exports what include/mf.h
declares; the binding refuses to run without a GPU; the per-event device code, compiled for the host by the
test-only shim tests/host_shim/, agrees with the oracle; the multi-rank sharding logic (gloo, world size 2).
"""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2106_10279_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
dp = C.POINTER(C.c_double)


# ---- the library and its header ---------------------------------------------------------------------------
@pytest.fixture(scope="module")
def libpath():
    from paper_2106_10279_b200 import build
    return build.build()     # nvcc cross-compiles without a GPU; no-op when up to date


def test_library_exports_every_declared_symbol(libpath):
    from paper_2106_10279_b200 import api
    hdr = open(os.path.join(ROOT, "include", "mf.h")).read()
    declared = sorted(set(re.findall(r"\b(mf_[a-z0-9_]+)\s*\(", hdr)))
    assert declared == sorted(api.EXPORTS)
    L = C.CDLL(libpath)
    for name in declared:
        assert hasattr(L, name), name


def test_struct_layouts_match_header():
    from paper_2106_10279_b200 import api
    assert C.sizeof(api.IterResult) == 40
    # int32 + pad, 9 doubles, 3 int32 + pad, 3 ptrs, int32 (pdf_nfl) + pad
    assert C.sizeof(api.ProcessDesc) == 8 + 9 * 8 + 4 + 4 + 4 + 4 + 3 * 8 + 8
    from oracle import mfo
    assert C.sizeof(mfo.ProcessDesc) == C.sizeof(api.ProcessDesc)
    assert [f[0] for f in mfo.ProcessDesc._fields_] == [f[0] for f in api.ProcessDesc._fields_]


def test_no_cpu_fallback(libpath):
    """Without a CUDA device the product path must fail loudly, not compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2106_10279_b200 import api
    with pytest.raises(api.MfError):
        api.Process(W.C0)
    d, keep = api.make_desc(W.C1, W.pdf_table())
    rc, h = api.mf_create_process(d)
    assert rc == api.MF_ECUDA and not h.value
    fl, ms = C.c_double(), C.c_double()
    assert api.lib().mf_measure_fp64_peak(1000, C.byref(fl), C.byref(ms)) != api.MF_OK


def test_product_does_not_import_oracle():
    """The CUDA path and the oracle share no code: neither includes nor imports the other."""
    pkg = os.path.join(ROOT, "paper_2106_10279_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle|#include\s+\"[^\"]*(oracle|mfo)", txt, re.M), f
                assert "libmfo" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".hpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2106_10279_b200" not in txt and "csrc" not in txt and "mf.h" not in txt.replace("include/mf.h", ""), f


# ---- device arithmetic compiled for the host (test-only shim) ----------------------------------------------
@pytest.fixture(scope="module")
def shim():
    src = os.path.join(ROOT, "tests", "host_shim", "mf_host_shim.cu")
    out = os.path.join(ROOT, "tests", "host_shim", "libmfh.so")
    from paper_2106_10279_b200 import build
    build.generate()
    deps = [src] + [os.path.join(build.CSRC, f) for f in os.listdir(build.CSRC)]
    if not os.path.exists(out) or any(os.path.getmtime(d) > os.path.getmtime(out) for d in deps):
        subprocess.check_call(["g++", "-x", "c++", "-std=c++17", "-O1", "-fPIC", "-shared", "-o", out, src])
    L = C.CDLL(out)
    L.mfh_me2.restype = C.c_double
    L.mfh_me2.argtypes = [C.c_int, dp, C.c_double, C.c_double, C.c_double]
    for f in (L.mfh_me2_coop, L.mfh_me2_coop3, L.mfh_me2_cta5, L.mfh_me2_qq_ttgg, L.mfh_me2_qq_ttgg_mem):
        f.restype = C.c_double
        f.argtypes = [dp, C.c_double, C.c_double]
    L.mfh_event.argtypes = [C.c_int, dp, C.c_int] + [C.c_double] * 8 + [C.c_uint64, C.c_uint32, C.c_uint64, dp]
    L.mfh_philox.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint32, C.POINTER(C.c_uint32)]
    L.mfh_uniform52.restype = C.c_double
    L.mfh_uniform52.argtypes = [C.c_uint32, C.c_uint32]
    L.mfh_me2_ttj_quark_classes.argtypes = [dp, C.c_double, C.c_double, dp]
    L.mfh_me2_light_line_ttg.restype = C.c_double
    L.mfh_me2_light_line_ttg.argtypes = [C.c_int, dp, C.c_double, C.c_double]
    for f in (L.mfh_pdf_2d, L.mfh_pdf_row, L.mfh_pdf_row_weights):
        f.restype = C.c_double
        f.argtypes = [dp, dp, dp, C.c_int, C.c_int, C.c_double, C.c_double]
    return L


def test_shim_philox_and_uniforms(shim):
    from oracle import mfo
    rng = np.random.default_rng(0)
    for _ in range(200):
        seed, it, ev, blk = (int(rng.integers(0, 2 ** 63)), int(rng.integers(0, 2 ** 32)), int(rng.integers(0, 2 ** 63)),
                             int(rng.integers(0, 2 ** 32)))
        out = (C.c_uint32 * 4)()
        shim.mfh_philox(seed, it, ev, blk, out)
        assert list(out) == mfo.philox_block(seed, it, ev, blk)
        assert shim.mfh_uniform52(out[0], out[1]) == mfo.uniform_from_words(out[0], out[1])


def test_shim_pdf_paths(shim, pdf, oracle_procs):
    lnx, lnq2, xf = pdf
    rng = np.random.default_rng(2)
    args = (lnx.ctypes.data_as(dp), lnq2.ctypes.data_as(dp), xf.ctypes.data_as(dp), len(lnx), len(lnq2))
    for _ in range(500):
        x = float(np.exp(rng.uniform(np.log(1e-8), 0)))
        q2 = float(np.exp(rng.uniform(np.log(3.0), np.log(9e9))))
        o = oracle_procs[1].pdf_xf(x, q2)
        assert abs(shim.mfh_pdf_2d(*args, x, q2) - o) <= 1e-12 * abs(o) + 1e-15
        # the collapsed-row path of the fused pass (Q^2 step applied to the knots first) is the same interpolant
        assert abs(shim.mfh_pdf_row(*args, x, q2) - o) <= 1e-11 * abs(o) + 1e-14
    # the multi-flavour pass forms the Hermite weights once per x: every table of the flavour set, ends included
    lnx, lnq2, xf = W.pdf_table_flavours()
    from oracle import mfo
    op = mfo.Process(W.C5, (lnx, lnq2, xf))
    xs = [1e-9, 1.0, float(np.exp(lnx[1])), float(np.exp(lnx[-2])), 0.999] + list(np.exp(rng.uniform(np.log(1e-8), 0, 200)))
    for t in range(xf.shape[0]):
        tab = np.ascontiguousarray(xf[t])
        args = (lnx.ctypes.data_as(dp), lnq2.ctypes.data_as(dp), tab.ctypes.data_as(dp), len(lnx), len(lnq2))
        scale = np.abs(tab).max(axis=1)
        for x in xs[:5] + xs[5 + 20 * t:25 + 20 * t]:
            q2 = float(np.exp(rng.uniform(np.log(3.0), np.log(9e9))))
            o = op.pdf_xf_table(t, x, q2)
            i = int(np.clip(np.searchsorted(lnx, np.log(x), side="right") - 1, 0, len(lnx) - 2))
            assert abs(shim.mfh_pdf_row_weights(*args, x, q2) - o) <= 1e-11 * abs(o) + 4e-15 * scale[max(i - 1, 0):i + 3].max()


@pytest.mark.parametrize("kind", [0, 1])
def test_shim_quark_gluon_channel_me(shim, kind):
    """q qbar -> ttbar g / q g -> ttbar q of the CUDA path's source against the oracle's Feynman-diagram sum"""
    from oracle import mfo
    rng = np.random.default_rng(10 + kind)
    mt = W.C2.m_top
    for _ in range(60):
        k, _ = mfo.rambo([mt, mt, 0.0], 400.0 + 3000.0 * rng.random(), rng.random(12))
        w = k[:, 0].sum() / 2
        mom = np.ascontiguousarray(np.vstack([[w, 0, 0, w], [w, 0, 0, -w], k]))
        g = shim.mfh_me2_light_line_ttg(kind, mom.ctypes.data_as(dp), mt, W.C2.alpha_s)
        o = mfo.me2_light_line_ttbar_g(kind, mom, mt, W.C2.alpha_s)
        assert abs(g / o - 1) < 1e-10, (g, o)


def test_shim_ttj_quark_classes_at_once(shim):
    """the six classes with shared top-line currents and native antiquark lines against the oracle's per-class diagram sums"""
    from oracle import mfo
    rng = np.random.default_rng(77)
    mt, a_s = W.C6.m_top, W.C6.alpha_s
    for _ in range(25):
        w = 400.0 + 4000.0 * rng.random() ** 2
        k, _ = mfo.rambo([mt, mt, 0.0], w, rng.random(12))
        mom = np.ascontiguousarray(np.vstack([[w / 2, 0, 0, w / 2], [w / 2, 0, 0, -w / 2], k]))
        out = np.zeros(6)
        shim.mfh_me2_ttj_quark_classes(mom.ctypes.data_as(dp), mt, a_s, out.ctypes.data_as(dp))
        sw = np.ascontiguousarray(mom[[1, 0, 2, 3, 4]])
        want = [mfo.me2_light_line_ttbar_g(0, mom, mt, a_s), mfo.me2_light_line_ttbar_g(0, sw, mt, a_s),
                mfo.me2_light_line_ttbar_g(1, mom, mt, a_s), mfo.me2_light_line_ttbar_g(1, sw, mt, a_s),
                mfo.me2_light_line_ttbar_g(2, mom, mt, a_s), mfo.me2_light_line_ttbar_g(2, sw, mt, a_s)]
        np.testing.assert_allclose(out, want, rtol=1e-11)


def test_shim_quark_channel_me(shim):
    """q qbar -> t tbar of the CUDA path's source (chiral two-component spinors) against the oracle (Dirac matrices)"""
    from oracle import mfo
    op = mfo.Process(W.C5, W.pdf_table_flavours())
    rng = np.random.default_rng(4)
    mt = W.C5.m_top
    for _ in range(200):
        E = mt * (1.0 + 10 ** rng.uniform(-4, 1.7))
        p = np.sqrt(E * E - mt * mt)
        ct, ph = rng.uniform(-1, 1), rng.uniform(0, 2 * np.pi)
        st = np.sqrt(1 - ct * ct)
        k = np.array([E, p * st * np.cos(ph), p * st * np.sin(ph), p * ct])
        mom = np.ascontiguousarray([[E, 0, 0, E], [E, 0, 0, -E], k, [E, -k[1], -k[2], -k[3]]])
        g = shim.mfh_me2(4, mom.ctypes.data_as(dp), mt, W.C5.alpha_s, W.C5.alpha_em)
        assert abs(g / op.me2_qq(mom) - 1) < 1e-11


@pytest.mark.parametrize("wl", [W.C0, W.C1, W.C2, W.C3], ids=["C0", "C1", "C2", "C3"])
def test_shim_event_chain(shim, wl, oracle_procs):
    """Philox -> VEGAS map -> phase space -> cuts -> |M|^2 of the CUDA path's source against the oracle."""
    op = oracle_procs[wl.process]
    n = 150 if wl.process < 3 else 60
    grid = W.uniform_grid(wl.n_dims)
    rows = op.debug_eval(grid, 0, 0, 0, n)
    D, nf = wl.n_dims, wl.n_final
    o = D + 4 * (nf + 2)
    ncut = nf - 2
    tau_min = ((2 * wl.m_top + ncut * wl.ptmin) ** 2 / wl.sqrt_s ** 2) if wl.process else 0.0
    npass = 0
    for e in range(n):
        out = np.zeros(64)
        shim.mfh_event(wl.process, grid.ctypes.data_as(dp), wl.n_bins, wl.sqrt_s, wl.m_top, wl.alpha_s, wl.alpha_em,
                       wl.ptmin, wl.etamax, wl.drmin, tau_min, 0, 0, e, out.ctypes.data_as(dp))
        r = rows[e]
        x1, x2, lum, me2, phi, jv, w, pas, rr = r[o:o + 9]
        assert out[5] == pas
        assert abs(out[0] - x1) <= 1e-13 * x1 and abs(out[1] - x2) <= 1e-13 * x2
        assert abs(out[2] - phi) <= 1e-12 * phi and abs(out[3] - jv) <= 1e-13 * jv
        assert np.array_equal(out[24:24 + D], r[o + 9 + D:o + 9 + 2 * D])
        if pas:
            npass += 1
            assert abs(out[6] - me2) <= 1e-11 * me2
    assert npass > n // 2


@pytest.mark.parametrize("pid,n", [(2, 3), (3, 4)])
def test_shim_cooperative_program(shim, oracle_procs, pid, n):
    """The cooperative programs of the fused pass (g g -> t tbar g: one warp per event; g g -> t tbar g g: 64
    threads; team threads emulated stage by stage on the host: S0, the table-driven phases, S4; top spin 0 only,
    doubled) against the oracle's full helicity sum."""
    from oracle import mfo
    rng = np.random.default_rng(5)
    fn = shim.mfh_me2_coop if n == 4 else shim.mfh_me2_coop3
    for i in range(40):
        w = 420.0 + 4000.0 * rng.random() ** 2
        k, _ = mfo.rambo([173.0, 173.0] + [0.0] * (n - 2), w, rng.random(4 * n))
        mom = np.ascontiguousarray(np.vstack([[w / 2, 0, 0, w / 2], [w / 2, 0, 0, -w / 2], k]))
        ref = oracle_procs[pid].me2(mom)
        got = fn(mom.ctypes.data_as(dp), 173.0, 0.118)
        assert abs(got - ref) <= 1e-11 * ref


def test_shim_five_gluon_block_program(shim, oracle_procs):
    """g g -> t tbar g g g (mf_me_cta5.cuh: one event per thread block, work items looped over stage by stage on the host;
    meet-in-the-middle amplitudes, top spin 0 doubled, plain colour loop instead of the DMMA tiles) against the oracle."""
    from oracle import mfo
    rng = np.random.default_rng(15)
    for i in range(6):
        w = 600.0 + 4000.0 * rng.random() ** 2
        k, _ = mfo.rambo([173.0, 173.0, 0.0, 0.0, 0.0], w, rng.random(20))
        mom = np.ascontiguousarray(np.vstack([[w / 2, 0, 0, w / 2], [w / 2, 0, 0, -w / 2], k]))
        ref = oracle_procs[6].me2(mom)
        got = shim.mfh_me2_cta5(mom.ctypes.data_as(dp), 173.0, 0.118)
        assert abs(got - ref) <= 1e-11 * ref, (i, got, ref)


def test_bench_flop_constants():
    """bench.py's roofline numerator: every literal is recomputed from the committed ncu metric logs, and the static
    matrix-element counts it reads are the generated headers' (the literals must not go stale silently)."""
    import importlib.util
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    b = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(b)
    for proc, path in b.FLOP_PROFILES.items():
        n, rate = b.FLOP_PROFILE_EVENTS[proc]
        total = b.executed_flops_of_profile(path)
        if proc in b.FLOP_PROFILE_ME:          # OTHER_FLOPS = (executed - n_pass x static count) / n
            other = (total - n * rate * b.FLOP_PROFILE_ME[proc]) / n
            assert abs(other - b.OTHER_FLOPS[proc]) <= 0.02 * b.OTHER_FLOPS[proc] + 10, (proc, other)
        else:                                   # measured total per (passing) event (+ the DMMA flop ncu's op counters miss)
            per = total / (n * rate) + b.FLOP_PROFILE_DMMA.get(proc, 0.0)
            assert abs(per - b.ME_FLOPS_MEASURED[proc]) <= 0.005 * per, (proc, per)
    from paper_2106_10279_b200 import build
    build.generate()
    for proc, (hdr, name) in b.FLOP_HEADERS.items():
        txt = open(os.path.join(build.CSRC, hdr)).read()
        assert ("constexpr double %s = %d.0;" % (name, b.me_flops(proc))) in txt
    # the static count of the profiled gg -> ttbar g build is still the header's (that kernel has not changed since)
    assert b.me_flops(2) == b.FLOP_PROFILE_ME[2]


def test_shim_qq_ttgg(shim):
    """the product's q qbar -> t tbar g g (13 + 13 currents, 20 colour strings, rank-11 colour form, left-handed light line doubled)
    against the oracle's 36 diagrams with explicit colour tensors at RAMBO points, both beam assignments"""
    from oracle import mfo
    rng = np.random.default_rng(21)
    mt, a_s = 173.0, 0.118
    for i in range(6):
        w = 500.0 + 3000.0 * rng.random()
        k, _ = mfo.rambo([mt, mt, 0.0, 0.0], w, rng.random(16))
        mom = np.vstack([[w / 2, 0, 0, w / 2], [w / 2, 0, 0, -w / 2], k])
        if i & 1:
            mom[[0, 1]] = mom[[1, 0]]
        want = mfo.me2_qq_ttbar_gg(mom, mt, a_s)
        for f in (shim.mfh_me2_qq_ttgg, shim.mfh_me2_qq_ttgg_mem):      # streamed top line; both lines' currents in memory
            assert f(np.ascontiguousarray(mom).ctypes.data_as(dp), mt, a_s) == pytest.approx(want, rel=1e-11)


# ---- multi-rank sharding (gloo, world size 2) ------------------------------------------------------------------
def test_shard_range_partitions():
    from paper_2106_10279_b200.integrate import shard_range
    for n in (0, 1, 7, 1 << 22, 10 ** 6 + 3):
        for world in (1, 2, 3, 8):
            nxt = 0
            for r in range(world):
                first, cnt = shard_range(n, r, world)
                assert first == nxt and cnt >= 0
                nxt = first + cnt
            assert nxt == n


_WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["MF_ROOT"])
import numpy as np, torch, torch.distributed as dist
from oracle import mfo
from paper_2106_10279_b200 import workloads as W
from paper_2106_10279_b200.integrate import shard_range, combine_across_ranks
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
wl, n = W.C1, 20001
op = mfo.Process(wl, W.pdf_table())
grid = W.uniform_grid(wl.n_dims)
for k in range(2):
    first, cnt = shard_range(n, rank, world)
    hist, res = op.vegas_iterate(grid, 0, k, first, cnt)        # the oracle stands in for the per-rank kernel
    r = torch.tensor(np.frombuffer(bytes(res), dtype=np.float64).copy())
    h = torch.from_numpy(hist.copy())
    combine_across_ranks(h, r)
    href, rref = op.vegas_iterate(grid, 0, k, 0, n)             # single-rank answer
    got = mfo.IterResult.from_buffer_copy(r.numpy().tobytes())
    assert got.n_pass == rref.n_pass and got.n_accept == rref.n_accept
    assert abs(got.sum_w - rref.sum_w) <= 1e-12 * abs(rref.sum_w)
    assert abs(got.sum_w2 - rref.sum_w2) <= 1e-12 * rref.sum_w2
    assert got.max_abs_w == rref.max_abs_w
    np.testing.assert_allclose(h.numpy(), href, rtol=1e-12)
    # every rank holds bit-identical totals, so the replicated refinement stays in lock-step
    mine = torch.cat([r, h.reshape(-1)])
    both = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(both, mine)
    assert all(torch.equal(both[0], b) for b in both)
    grid = op.refine_grid(grid, h.numpy(), W.VEGAS_ALPHA)
dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_two_rank_iteration_gloo(tmp_path):
    """Shard -> per-rank sums -> one all-gather -> fixed-order combine equals the single-rank iteration."""
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, MF_ROOT=ROOT, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
           "127.0.0.1", "--master-port", "29533", str(script)]
    r = subprocess.run(cmd, env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-3000:]
    assert r.stdout.count("ok") >= 2


def test_combined_estimate():
    from paper_2106_10279_b200.integrate import IterationRecord, RunResult
    rr = RunResult()
    # two iterations with known I, sigma: I = sum_w/n ; sigma^2 = (sum_w2/n - I^2)/(n-1)
    n = 1001
    for I, s in ((2.0, 0.1), (2.2, 0.2)):
        sum_w2 = (s * s * (n - 1) + I * I) * n
        rr.iterations.append(IterationRecord(0, n, I * n, sum_w2, 0.0, n, 0))
    mean, err, chi2 = rr.combined()
    w1, w2 = 1 / 0.01, 1 / 0.04
    assert abs(mean - (2.0 * w1 + 2.2 * w2) / (w1 + w2)) < 1e-9
    assert abs(err - (w1 + w2) ** -0.5) < 1e-9
    assert abs(chi2 - ((2.0 - mean) ** 2 * w1 + (2.2 - mean) ** 2 * w2)) < 1e-7
