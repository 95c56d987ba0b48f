"""CPU-only checks of the boundary: libra.so loads, exports every symbol include/ra.h declares, the planner
(host logic of S3) behaves, argument errors are reported before any CUDA call, and nothing in the product
imports the oracle."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def ra():
    import paper_2606_09200_b200 as m
    return m


def _header_functions():
    src = open(os.path.join(ROOT, "include", "ra.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ra_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(ra):
    lib = ctypes.CDLL(ra.lib_path())
    names = _header_functions()
    assert {"ra_gemm", "ra_allreduce_emul", "ra_alltoall_emul", "ra_overlap_run"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(ra.EXPORTS) == names            # the binding covers exactly the header


def test_status_strings(ra):
    assert [ra.status_str(i) for i in range(6)] == ["RA_OK", "RA_ERR_INVALID_ARG", "RA_ERR_UNSUPPORTED",
                                                     "RA_ERR_INFEASIBLE_KNOB", "RA_ERR_CUDA", "RA_ERR_ARCH"]


def test_struct_layouts_match_header(ra):
    # sizes computed by hand from include/ra.h (LP64)
    assert ctypes.sizeof(ra.Occupancy) == 40
    assert ctypes.sizeof(ra.GemmPlan) == 72
    assert ctypes.sizeof(ra.Workload) == 160
    assert ctypes.sizeof(ra.OverlapCfg) == 4 + 40 + 9 * 4
    assert ctypes.sizeof(ra.OverlapResult) == 24 + 72 + 8
    assert ctypes.sizeof(ra.HostIO) == 7 * 8


KB = 1024


@pytest.mark.parametrize("shape", [(8192, 8192, 8192), (64, 16384, 16384), (256, 256, 256), (200, 136, 72)])
@pytest.mark.parametrize("reserve", [0, 32 * KB, 64 * KB, 96 * KB, 128 * KB, 160 * KB, 200 * KB])
@pytest.mark.parametrize("budget", [0, 74, 110, 148])
def test_plan_honours_reserve_and_budget(ra, shape, reserve, budget):
    M, N, K = shape
    p = ra.ra_gemm_plan_query(0, 1, M, N, K, dict(smem_reserve_bytes=reserve, sm_budget=budget))
    # S3: the GEMM leaves the reserve unallocated on every SM, under the residency the plan accounts for -- which is
    # what the hardware admits (hw_ctas_per_sm) unless padding excludes the second CTA.  Only a reserve that not even
    # two one-stage CTAs fit under (200 KiB) is clamped, and says so.
    assert p["smem_left_per_sm"] >= reserve or (p["clamped"] == 1 and reserve == 200 * KB), p
    assert p["ctas_per_sm"] == p["hw_ctas_per_sm"] or p["clamped"], p
    assert p["smem_left_per_sm"] == 228 * KB - p["ctas_per_sm"] * (p["dyn_smem_bytes"] + KB), p
    if reserve <= 112 * KB:
        assert p["ctas_per_sm"] == 1 and 2 * (p["dyn_smem_bytes"] + KB) > 228 * KB, p     # a second CTA cannot fit
    assert p["stages"] >= 1 and p["tile_k"] == 64
    assert p["grid"] <= (budget or 148)
    assert p["dyn_smem_bytes"] <= 227 * KB
    tiles = -(-M // p["tile_m"]) * -(-N // p["tile_n"])
    assert p["n_tiles"] == tiles
    ws = ra.ra_gemm_workspace_bytes(0, 1, M, N, K, dict(smem_reserve_bytes=reserve, sm_budget=budget))
    assert (ws > 0) == (p["split_k"] > 1)


def test_plan_depth_shrinks_with_reserve(ra):
    stages = [ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192, dict(smem_reserve_bytes=r * KB))["stages"] for r in (0, 64, 112)]
    assert stages == sorted(stages, reverse=True) and stages[0] == 4          # big tiles: 4 x 48 KiB
    p0 = ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192)
    assert p0["m_blocks"] == 2 and p0["tile_m"] == 512 and p0["cta_group"] == 2 and p0["n_tiles"] == 512
    p1 = ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192, dict(m_blocks=1))
    assert p1["m_blocks"] == 1 and p1["tile_m"] == 256 and p1["stages"] == 6     # 6 x 32 KiB + 32 KiB store staging
    # too little shared memory for three 48 KiB stages -> back to one block per CTA
    p2 = ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192, dict(smem_reserve_bytes=112 * KB))
    assert p2["m_blocks"] == 1 and p2["smem_left_per_sm"] >= 112 * KB
    mb = [ra.ra_gemm_plan_query(0, 1, 64, 16384, 16384, dict(smem_reserve_bytes=r * KB)) for r in (0, 64, 128, 200)]
    assert [p["stages"] for p in mb] == sorted((p["stages"] for p in mb), reverse=True)
    assert all(p["swap_ab"] == 1 and p["tile_m"] == 64 for p in mb)
    assert mb[0]["split_k"] == 1 and mb[0]["grid"] == 128           # one tile per CTA on 128 of the 148 SMs
    for b in (74, 92, 110):                                         # ragged multi-wave -> stream-K on exactly b CTAs
        p = ra.ra_gemm_plan_query(0, 1, 64, 16384, 16384, dict(sm_budget=b))
        assert p["split_k"] > 1 and p["grid"] == b


def test_cluster_split_k_plans(ra):
    p = ra.ra_gemm_plan_query(0, 1, 8192, 64, 8192)                   # 64 single-CTA tiles, long K: picked automatically
    assert p["cluster_k"] == 2 and p["grid"] == 128 and p["split_k"] == 1
    assert ra.ra_gemm_workspace_bytes(0, 1, 8192, 64, 8192) == 0
    assert ra.ra_gemm_plan_query(0, 1, 8192, 64, 8192, dict(cluster_k=1))["cluster_k"] == 1
    # not available for CTA-pair tiles or in bounded-work mode: clamped, or refused without allow_clamp
    p4 = ra.ra_gemm_plan_query(0, 1, 128, 1024, 16384)               # 8 weight tiles, 256 k-blocks: four parts per tile
    assert p4["cluster_k"] == 4 and p4["grid"] == 32 and ra.ra_gemm_workspace_bytes(0, 1, 128, 1024, 16384) == 0
    for occ in (dict(cluster_k=2, m_blocks=2), dict(cluster_k=2, tiles_per_cta=1)):
        q = ra.ra_gemm_plan_query(0, 1, 2048, 2048, 2048, occ)
        assert q["cluster_k"] == 1 and q["clamped"] == 1, q
        with pytest.raises(ra.RaError) as e:
            ra.ra_gemm_plan_query(0, 1, 2048, 2048, 2048, dict(occ, allow_clamp=0))
        assert e.value.status == ra.RA_ERR_INFEASIBLE_KNOB


def test_small_problem_takes_one_narrow_wave(ra):
    p = ra.ra_gemm_plan_query(0, 1, 1024, 1024, 1024)
    assert (p["tile_m"], p["tile_n"], p["grid"], p["split_k"], p["cta_group"]) == (128, 64, 128, 1, 1), p
    p = ra.ra_gemm_plan_query(0, 1, 256, 256, 256)
    assert (p["tile_n"], p["grid"]) == (64, 8), p
    assert ra.ra_gemm_plan_query(0, 1, 2048, 2048, 2048)["cta_group"] == 2      # too big for one wave: pair tiles


def test_plan_infeasible_knob(ra):
    with pytest.raises(ra.RaError) as e:
        ra.ra_gemm_plan_query(0, 1, 512, 512, 512, dict(smem_reserve_bytes=226 * KB, allow_clamp=0))
    assert e.value.status == ra.RA_ERR_INFEASIBLE_KNOB
    p = ra.ra_gemm_plan_query(0, 1, 512, 512, 512, dict(smem_reserve_bytes=226 * KB, allow_clamp=1))
    assert p["clamped"] == 1 and p["stages"] == 1
    with pytest.raises(ra.RaError):
        ra.ra_gemm_plan_query(0, 1, 512, 512, 512, dict(sm_budget=1000, allow_clamp=0))
    assert ra.ra_gemm_plan_query(0, 1, 512, 512, 512, dict(sm_budget=1000))["clamped"] == 1


def test_bounded_work_mode_grid(ra):
    p = ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192, dict(tiles_per_cta=4))
    assert p["n_tiles"] == 512 and p["cta_group"] == 2                # 512 x 256 tiles on CTA pairs
    assert p["grid"] == 2 * 512 // 4 and p["split_k"] == 1            # 2 CTAs per tile, 4 tiles per pair
    assert 2 * (p["dyn_smem_bytes"] + 1024) > 228 * KB               # a second GEMM CTA cannot fit on the SM


def test_argument_errors_need_no_gpu(ra):
    fake = 0x10000
    lib = ra._L()
    P = ctypes.POINTER(ctypes.c_void_p)
    arr = (ctypes.c_void_p * 2)(fake, fake + 4096)
    assert lib.ra_allreduce_emul(None, 2, 16, 0, None) == ra.RA_ERR_INVALID_ARG
    assert lib.ra_allreduce_emul(arr, 0, 16, 0, None) == ra.RA_ERR_INVALID_ARG
    assert lib.ra_allreduce_emul(arr, 2, 4096, 0, None) == ra.RA_ERR_INVALID_ARG        # buffers overlap
    assert lib.ra_allreduce_emul((ctypes.c_void_p * 2)(fake + 4, fake + 4096), 2, 16, 0, None) == ra.RA_ERR_INVALID_ARG
    assert lib.ra_allreduce_emul(arr, 2, 0, 0, None) == ra.RA_OK                        # count == 0: nothing to do
    assert lib.ra_alltoall_emul(fake, fake + 64, 2, 64, 0, None) == ra.RA_ERR_INVALID_ARG  # overlap
    assert lib.ra_alltoall_emul(fake, fake + 4096, 2, 24, 0, None) == ra.RA_ERR_INVALID_ARG
    assert lib.ra_alltoall_emul(fake, fake + 4096, 2, 0, 0, None) == ra.RA_OK
    g = dict(transA=0, transB=1, M=32, N=32, K=64, alpha=1.0, A=fake, lda=64, B=fake + (1 << 20), ldb=64, beta=0.0,
             C=fake + (2 << 20), ldc=32)
    for kw, st in [(dict(M=-1), 1), (dict(transA=2), 1), (dict(A=None), 1), (dict(lda=8), 1), (dict(ldc=24), 1),
                   (dict(ldc=36), 2), (dict(A=fake + 2), 1), (dict(transB=0, ldb=24), 1), (dict(transA=1, lda=24), 1), (dict(M=0), 0)]:
        a = dict(g, **kw)
        s = lib.ra_gemm(a["transA"], a["transB"], a["M"], a["N"], a["K"], a["alpha"], a["A"], a["lda"], a["B"], a["ldb"],
                        a["beta"], a["C"], a["ldc"], None, None, 0, None)
        assert s == st, (kw, s)
    assert lib.ra_overlap_run(None, None, None) == ra.RA_ERR_INVALID_ARG


def test_overlap_driver_validates_the_collective_before_touching_it(ra):
    """A bad collective description is RA_ERR_INVALID_ARG from ra_overlap_run / _run_host / _sweep: no pointer array is
    read past P, nothing is enqueued (ra.h: 'a failing call has no side effects').  Needs no device."""
    lib = ra._L()
    fake = 0x100000
    g = dict(M=128, N=128, K=128, A=fake, B=fake + (1 << 20), C=fake + (2 << 20))
    bufs = [_FakeBuf(1024, fake + (4 << 20) + i * 8192) for i in range(4)]
    res = ra.OverlapResult()

    def run(w, **kw):
        return lib.ra_overlap_run(ctypes.byref(w), ctypes.byref(ra.make_cfg(**kw)), ctypes.byref(res))

    w, keep = ra.make_workload(gemm=g, allreduce=bufs, n_iters=2)
    w.ar_bufs = None
    assert run(w) == ra.RA_ERR_INVALID_ARG                                    # NULL pointer array (was a host segfault)
    for bad_p in (0, -3, ra.RA_MAX_RANKS + 1, 1 << 20):
        w, keep = ra.make_workload(gemm=g, allreduce=bufs, n_iters=2)
        w.P = bad_p
        assert run(w) == ra.RA_ERR_INVALID_ARG, bad_p
        assert run(w, use_graph=1) == ra.RA_ERR_INVALID_ARG, bad_p            # the graph key must not read ar_bufs[0..P)
    w, keep = ra.make_workload(gemm=g, allreduce=[_FakeBuf(1024, fake), _FakeBuf(1024, fake + 2048)], n_iters=2)
    assert run(w) == ra.RA_ERR_INVALID_ARG                                    # rank buffers overlap
    w, keep = ra.make_workload(gemm=g, allreduce=bufs, n_iters=2, ar_pristine=[bufs[1]] * 4)
    assert run(w) == ra.RA_ERR_INVALID_ARG                                    # pristine copy aliases a rank buffer
    w, keep = ra.make_workload(gemm=g, allreduce=bufs, n_iters=2)
    assert run(w, coll_variant=1, coll_smem_bytes=64) == ra.RA_ERR_INVALID_ARG   # ring too small for one slice
    for a2a in (dict(a=None, b=fake, P=2, chunk_bytes=64), dict(a=fake, b=fake + 64, P=2, chunk_bytes=64),
                dict(a=fake, b=fake + 4096, P=2, chunk_bytes=24), dict(a=fake, b=fake + 4096, P=0, chunk_bytes=64),
                dict(a=fake + 8, b=fake + 4096, P=2, chunk_bytes=64)):
        w, keep = ra.make_workload(gemm=g, alltoall=a2a, n_iters=2)
        assert run(w) == ra.RA_ERR_INVALID_ARG, a2a
    w, keep = ra.make_workload(gemm=g, alltoall=dict(a=fake, b=fake + 4096, P=2, chunk_bytes=64), n_iters=2)
    assert run(w, coll_variant=7) == ra.RA_ERR_INVALID_ARG
    # host-buffer entry point: P is checked before io->ar_in[0..P) is indexed
    w, keep = ra.make_workload(gemm=g, allreduce=bufs, n_iters=2)
    w.P = 1 << 20
    io, keep_io = ra.make_host_io(A=fake, B=fake, ar_in=[fake] * 4)
    assert lib.ra_overlap_run_host(ctypes.byref(w), None, ctypes.byref(io), ctypes.byref(ra.make_cfg()), 1,
                                   ctypes.byref(res)) == ra.RA_ERR_INVALID_ARG
    cfgs = (ra.OverlapCfg * 1)(ra.make_cfg())
    best = ctypes.c_int(-1)
    assert lib.ra_overlap_sweep(ctypes.byref(w), cfgs, 1, 3, (ra.OverlapResult * 1)(), ctypes.byref(best)) == ra.RA_ERR_INVALID_ARG


def test_compute_fails_loudly_without_device(ra):
    try:
        import torch
        if torch.cuda.is_available():
            pytest.skip("GPU present")
    except ImportError:
        pass
    arr = (ctypes.c_void_p * 2)(0x10000, 0x20000)
    s = ra._L().ra_allreduce_emul(arr, 2, 16, 0, None)
    assert s in (ra.RA_ERR_CUDA, ra.RA_ERR_ARCH)                    # no CPU fallback
    assert ra.status_str(s).startswith("RA_ERR")


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2606_09200_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "liboracle" not in txt and "oracle.c" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_09200_b200" not in txt and "ra.h" not in txt


# ---- S7': the model-based knob policy is host-only, so its logic is tested here ---------------------------------------
class _FakeBuf:
    def __init__(self, n, ptr=16):
        self.n = n
        self.ptr = ptr

    def numel(self):
        return self.n

    def data_ptr(self):
        return self.ptr


def _workload(ra, M, N, K, coll, P, count=0, chunk=0, n_iters=20):
    g = dict(M=M, N=N, K=K, A=16, B=16, C=16)
    if coll == "allreduce":
        return ra.make_workload(gemm=g, allreduce=[_FakeBuf(count) for _ in range(P)], n_iters=n_iters)
    return ra.make_workload(gemm=g, alltoall=dict(a=16, b=32, P=P, chunk_bytes=chunk), n_iters=n_iters)


def test_policy_rooflines_and_choices(ra):
    T, H = 1400.0, 6450.0
    # compute-bound GEMM + allreduce: tensor roofline, all SMs, no reserve, priority off
    w, keep = _workload(ra, 8192, 8192, 8192, "allreduce", 8, count=16 << 20)
    s = ra.ra_overlap_suggest(w, T, H)
    flops, gb, cb = 2.0 * 8192 ** 3, 2.0 * 3 * 8192 ** 2, 2.0 * 4 * 8 * (16 << 20)
    eff = 512 / (7 * 74)                                      # 512 big tiles on 74 CTA pairs: 7 waves
    assert s["gemm_bound"] == "tensor"
    assert abs(s["t_gemm_ms"] - flops / (T * 1e9 * eff)) < 1e-9
    assert abs(s["t_coll_ms"] - cb / (H * 1e6)) < 1e-9
    assert abs(s["t_roofline_ms"] - max(s["t_gemm_ms"], (gb + cb) / (H * 1e6))) < 1e-9
    assert abs(s["t_serial_ms"] - (s["t_gemm_ms"] + s["t_coll_ms"])) < 1e-12
    assert s["t_gemm_ms"] <= s["t_overlap_ms"] <= s["t_serial_ms"]
    kw = s["kw"]
    assert kw["occ"]["sm_budget"] == 0 and kw["occ"]["smem_reserve_bytes"] == 0 and kw["prio_comm"] == kw["prio_compute"]
    assert kw["coll_variant"] == 0                              # tensor-bound GEMM: the register allreduce co-resides everywhere
    # the same GEMM under a collective seven times larger (the paper's literal cb-ar): the collective is the long pole,
    # so the GEMM gives up a pipeline stage (32 KiB reserve) to leave the co-resident collective its L1
    wl, keepl = _workload(ra, 8192, 8192, 8192, "allreduce", 4, count=224 << 20, n_iters=10)
    sl = ra.ra_overlap_suggest(wl, T, H)
    assert sl["kw"]["occ"]["smem_reserve_bytes"] == 32 * KB and sl["t_coll_ms"] > sl["t_gemm_ms"]
    wl, keepl = _workload(ra, 8192, 8192, 8192, "alltoall", 4, chunk=224 << 20, n_iters=10)
    sl = ra.ra_overlap_suggest(wl, T, H)
    assert sl["kw"]["coll_variant"] == 2 and sl["kw"]["occ"]["smem_reserve_bytes"] == 0     # copy engines: no SM resource at all
    # the same GEMM fills shared memory, so the alltoall must be the shared-memory-free variant
    w, keep = _workload(ra, 8192, 8192, 8192, "alltoall", 8, chunk=8 << 20)
    assert ra.ra_overlap_suggest(w, T, H)["kw"]["coll_variant"] == 1
    # skinny GEMM + allreduce: the TMA-ring allreduce (variant 1) on the SMs the GEMM leaves free
    w, keep = _workload(ra, 64, 16384, 16384, "allreduce", 8, count=16 << 20)
    assert ra.ra_overlap_suggest(w, T, H)["kw"]["coll_variant"] == 1
    # skinny GEMM: HBM-bound, leaves 20 SMs free -> TMA-ring alltoall; overlap cannot beat total bytes / bandwidth
    w, keep = _workload(ra, 64, 16384, 16384, "alltoall", 8, chunk=8 << 20)
    s = ra.ra_overlap_suggest(w, T, H)
    gb = 2.0 * (64 * 16384 + 16384 * 16384 + 64 * 16384)
    assert s["gemm_bound"] == "hbm" and s["kw"]["coll_variant"] == 0
    assert abs(s["t_roofline_ms"] - (gb + float(1 << 30)) / (H * 1e6)) < 1e-9
    assert abs(s["t_overlap_ms"] - s["t_serial_ms"]) < 1e-9     # bytes-bound on both sides: nothing to hide
    assert s["kw"]["use_graph"] == 0                             # full-size kernels: nothing launch-bound to capture
    wt, keept = _workload(ra, 256, 256, 256, "allreduce", 4, count=65536, n_iters=4)
    assert ra.ra_overlap_suggest(wt, T, H)["kw"]["use_graph"] == 1     # Tiny: microsecond kernels -> CUDA-graph replay
    # one pipelined iteration has no partner for either kernel: the prediction is the serial time
    w, keep = _workload(ra, 8192, 8192, 8192, "allreduce", 8, count=16 << 20, n_iters=1)
    s = ra.ra_overlap_suggest(w, T, H)
    assert abs(s["t_overlap_ms"] - s["t_serial_ms"]) < 1e-9


def test_policy_budget_follows_wave_quantisation(ra):
    # 4096 x 4608: 8 x 18 = 144 big tiles -> 72 pairs run them in 2 full waves (eff 1.0), 74 pairs need 2 waves at 97 %:
    # the model must not pick a budget that quantises worse than all SMs, and must pick an even count
    w, keep = _workload(ra, 4096, 4608, 8192, "allreduce", 8, count=1 << 20)
    s = ra.ra_overlap_suggest(w)
    b = s["kw"]["occ"]["sm_budget"]
    assert b % 2 == 0 and (b == 0 or 74 <= b <= 148)
    p_all = ra.ra_gemm_plan_query(0, 1, 4096, 4608, 8192)
    p_pick = ra.ra_gemm_plan_query(0, 1, 4096, 4608, 8192, dict(sm_budget=b))

    def t(p):
        workers = p["grid"] // p["cta_group"]
        waves = -(-p["n_tiles"] // workers)
        return 1.0 / ((p["grid"] / 148) * (p["n_tiles"] / (waves * workers)))
    assert t(p_pick) <= t(p_all) * 1.0001


def test_policy_errors(ra):
    import ctypes
    lib = ctypes.CDLL(ra.lib_path())
    assert lib.ra_overlap_suggest(None, None, None) == ra.RA_ERR_INVALID_ARG


def test_header_is_plain_c_and_links_from_c(ra, tmp_path):
    """include/ra.h is the boundary: it must compile as C99 without any CUDA or C++ header, and a plain C program
    linked against libra.so must be able to call the host-only entry points."""
    import subprocess
    src = tmp_path / "use_ra.c"
    src.write_text(
        '#include "ra.h"\n#include <stdio.h>\n'
        "int main(void) {\n"
        "  ra_gemm_plan p; ra_occupancy o = {0, 0, 0, 1, 0, 0, 0, 0, 0, 0};\n"
        "  if (ra_gemm_plan_query(0, 1, 8192, 8192, 8192, &o, &p) != RA_OK) return 1;\n"
        '  printf("%d %d %d %s\\n", p.tile_m, p.tile_n, p.grid, ra_status_str(RA_ERR_ARCH));\n'
        "  return ra_gemm_plan_query(0, 1, 8, 8, 8, &o, (ra_gemm_plan*)0) == RA_ERR_INVALID_ARG ? 0 : 2;\n"
        "}\n")
    exe = tmp_path / "use_ra"
    libdir = os.path.dirname(ra.lib_path())
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"), str(src),
                           "-o", str(exe), "-L", libdir, "-l:libra.so", "-Wl,-rpath," + libdir])
    out = subprocess.check_output([str(exe)]).decode().split()
    assert out == ["512", "256", "148", "RA_ERR_ARCH"]


# ---- planner invariants over random shapes and knobs (host only) -------------------------------------------------
def test_planner_invariants_random(ra):
    from hypothesis import given, settings, strategies as st

    dims = st.one_of(st.integers(1, 300), st.sampled_from([64, 128, 256, 512, 1024, 4096, 8192, 16384, 57344]))
    occs = st.fixed_dictionaries(dict(
        smem_reserve_bytes=st.sampled_from([0, 0, 0, 32 * KB, 64 * KB, 96 * KB, 128 * KB, 160 * KB, 200 * KB]),
        sm_budget=st.sampled_from([0, 0, 0, 1, 2, 9, 33, 74, 92, 110, 128, 140, 148]),
        tiles_per_cta=st.sampled_from([0, 0, 0, 1, 2, 4]), cta_group=st.sampled_from([0, 0, 1, 2]),
        m_blocks=st.sampled_from([0, 0, 1, 2]), cluster_k=st.sampled_from([0, 0, 1, 2, 4]),
        l2_persist_bytes=st.sampled_from([0, 0, 0, 15 << 20, 47 << 20, 79 << 20]), tile_k=st.sampled_from([0, 0, 32, 64]),
        tile_order=st.sampled_from([0, 0, 1])))

    @settings(max_examples=400, deadline=None)
    @given(dims, dims, dims, st.integers(0, 1), st.integers(0, 1), occs)
    def prop(M, N, K, tA, tB, occ):
        p = ra.ra_gemm_plan_query(tA, tB, M, N, K, occ)          # allow_clamp = 1: never refuses a valid shape
        budget = occ["sm_budget"] or 148
        assert p["grid"] >= 1 and p["stages"] >= 1 and p["tile_k"] in (32, 64)
        # tile_k = 32 only where asked for AND applicable (K-contiguous operands, no cluster split-K); never silently
        assert (p["tile_k"] == 32) == (occ["tile_k"] == 32 and tA == 0 and tB == 1 and occ["cluster_k"] < 2), p
        if occ["tile_k"] == 32 and p["tile_k"] == 64:
            assert p["clamped"] == 1
        # the raster and the L2 knob: groups are at least one tile row wide; the knob is reported only where it is used,
        # and using it never changes the tile, the grid or the pipeline
        assert 1 <= p["group_x"] <= max(1, -(-(N if p["swap_ab"] else M) // (p["tile_n"] if p["swap_ab"] else p["tile_m"])))
        assert p["l2_persist_bytes"] in (0, occ["l2_persist_bytes"])
        if occ["l2_persist_bytes"]:
            q = ra.ra_gemm_plan_query(tA, tB, M, N, K, dict(occ, l2_persist_bytes=0))
            assert {k: v for k, v in p.items() if k not in ("group_x", "l2_persist_bytes")} == \
                   {k: v for k, v in q.items() if k not in ("group_x", "l2_persist_bytes")}
        # tile_order is a run-time choice: it never changes the plan
        assert ra.ra_gemm_plan_query(tA, tB, M, N, K, dict(occ, tile_order=1 - occ["tile_order"])) == p
        assert p["dyn_smem_bytes"] <= 227 * KB
        assert p["clamped"] or p["smem_left_per_sm"] >= occ["smem_reserve_bytes"], p
        assert p["n_tiles"] == -(-M // p["tile_m"]) * -(-N // p["tile_n"]), p
        assert p["cta_group"] in (1, 2) and p["m_blocks"] in (1, 2) and p["cluster_k"] in (1, 2, 4)
        if p["m_blocks"] == 2:
            assert p["cta_group"] == 2 and p["tile_m"] == 512
        per_tile = p["cta_group"] * p["cluster_k"]
        assert p["grid"] % per_tile == 0
        if occ["tiles_per_cta"] == 0:
            assert p["grid"] <= budget or p["clamped"], p            # persistent: at most one CTA per budgeted SM
        if p["cluster_k"] > 1:
            assert p["grid"] == per_tile * p["n_tiles"] and p["split_k"] == 1, p
        ws = ra.ra_gemm_workspace_bytes(tA, tB, M, N, K, occ)
        assert (ws > 0) == (p["split_k"] > 1), p
        if occ["cta_group"] == 1:
            assert p["cta_group"] == 1
        if occ["cluster_k"] == 1:
            assert p["cluster_k"] == 1

    prop()


def test_l2_persist_plan(ra):
    """occ.l2_persist_bytes: the raster group is widened to the X panel the carve-out holds (equal groups), the plan
    reports the knob only where it is used, and everything else about the plan is unchanged (a
    resource knob, not a different algorithm)."""
    base = ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192)
    assert base["group_x"] == 6 and base["l2_persist_bytes"] == 0
    p = ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192, dict(l2_persist_bytes=79 << 20))
    assert p["group_x"] == 8 and p["l2_persist_bytes"] == 79 << 20            # 9 panels of 8 MiB fit: 16 rows -> 8 + 8
    assert {k: v for k, v in p.items() if k not in ("group_x", "l2_persist_bytes")} == \
           {k: v for k, v in base.items() if k not in ("group_x", "l2_persist_bytes")}
    q = ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192, dict(l2_persist_bytes=32 << 20))
    assert q["group_x"] == 6 and q["l2_persist_bytes"] == 32 << 20            # smaller than the default group: keeps part of it
    # swapped (skinny), single-wave and stream-K plans ignore the knob
    assert ra.ra_gemm_plan_query(0, 1, 64, 16384, 16384, dict(l2_persist_bytes=79 << 20))["l2_persist_bytes"] == 0
    assert ra.ra_gemm_plan_query(0, 1, 2048, 2048, 2048, dict(l2_persist_bytes=79 << 20))["l2_persist_bytes"] == 0
    with pytest.raises(ra.RaError):
        ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192, dict(l2_persist_bytes=-1))
    for bad in (dict(tile_order=2), dict(tile_order=-1), dict(tile_k=16)):
        with pytest.raises(ra.RaError):
            ra.ra_gemm_plan_query(0, 1, 8192, 8192, 8192, bad)
