"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol include/ugks.h declares,
argument validation that happens before any CUDA call, and the rank plumbing of bench.py under gloo (world size 2)."""
import ctypes as C
import json
import os
import re
import subprocess
import sys

import numpy as np
import pytest

import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libugks():
    from paper_1810_08137_b200 import build
    build.build()
    from paper_1810_08137_b200 import binding
    return binding.lib()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "ugks.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ugks_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(libugks):
    from paper_1810_08137_b200 import binding
    names = _declared_functions()
    assert len(names) >= 17 and "ugks_step" in names and "ugks_residual" in names
    for n in names:
        assert hasattr(libugks, n), n
    assert sorted(binding.EXPORTS) == names


def test_version_and_workspace_bytes(libugks):
    from paper_1810_08137_b200 import binding
    assert b"sm_100a" in libugks.ugks_version()
    p = workloads.channel_config("C1")
    nb = binding.workspace_bytes(p)
    assert nb >= 2 * p.points * 8 and nb < 2 * p.points * 8 + (8 << 20)       # two copies of f + small per-face / per-cell arrays
    p4 = workloads.channel_config("C4")
    assert binding.workspace_bytes(p4) < 17e9                                # C4: 13.4 GB of f + 2.5 GB of per-face / per-cell records
    bad = workloads.channel_config("C1", I=1)
    assert binding.workspace_bytes(bad) == 0
    # velocity grids: up to 512 columns (one thread per column of a CTA), not more
    import dataclasses
    for nu, ok in ((256, True), (512, True), (513, False)):                  # (Nv = 16 here)
        u, wu = workloads.trapezoid_grid(nu, 20.0)
        q = dataclasses.replace(workloads.channel_config("C1"), u=u, wu=wu)
        assert (binding.workspace_bytes(q) > 0) == ok, nu


def test_argument_validation_happens_before_cuda(libugks):
    """EINVAL paths return before the library touches the device, so they can be checked here."""
    from paper_1810_08137_b200 import binding
    p = workloads.channel_config("C1")
    keep, mesh, vg, gas, bcs = binding._structs(p)
    h = C.c_void_p()
    ws = C.c_void_p(256)                                                      # never dereferenced on these paths

    def init(mesh=mesh, vg=vg, gas=gas, bcs=bcs, cfl=0.8, ws=ws, nbytes=1 << 40):
        return libugks.ugks_init(C.byref(h), C.byref(mesh), C.byref(vg), C.byref(gas), C.byref(bcs), cfl, ws, nbytes, None)

    g2 = binding._Gas(gas.omega, gas.mu_ref, gas.Kn, 2.0 / 3.0, 0)
    assert init(gas=g2) == 1 and b"Pr" in libugks.ugks_last_error(None)
    g3 = binding._Gas(gas.omega, gas.mu_ref, gas.Kn, 1.0, 2)
    assert init(gas=g3) == 1 and b"K_int" in libugks.ugks_last_error(None)
    assert init(cfl=0.0) == 1
    b2 = binding._BCs(bcs.xmin, bcs.xmax, binding._BC(0, 1, 0, 0, 1), bcs.ymax)
    assert init(bcs=b2) == 1 and b"periodic" in libugks.ugks_last_error(None)
    assert init(nbytes=16) == 2                                               # UGKS_ENOMEM
    assert init(ws=C.c_void_p(8)) == 1                                        # misaligned workspace
    assert libugks.ugks_step(None, 1) == 1 and libugks.ugks_sync(None) == 1
    assert libugks.ugks_dt(None) == 0.0 and libugks.ugks_step_count(None) == -1


def test_velocity_grid_limits_and_non_finite_nodes(libugks):
    """(1) a grid whose nodes, weights and chunk table overflow the 64 KB constant bank of the run-time compiled kernels
    is refused by ugks_workspace_bytes already (it used to pass there and fail in NVRTC at ugks_init); the largest accepted
    shapes do compile.  (2) NaN / Inf nodes or weights are UGKS_EINVAL before anything is compiled."""
    import dataclasses
    from paper_1810_08137_b200 import binding
    base = workloads.channel_config("C1", I=8, J=4)

    def grid(nu, nv):
        u, wu = workloads.trapezoid_grid(nu, 20.0)
        v, wv = workloads.trapezoid_grid(nv, 20.0)
        return dataclasses.replace(base, u=u, wu=wu, v=v, wv=wv)

    assert binding.workspace_bytes(grid(8, 2049)) == 0                        # Nv <= 2048
    assert binding.workspace_bytes(grid(512, 2048)) == 0                      # 1-row chunks: 2048 x 16 B of chunk table on top of 40 KB of nodes
    for nu, nv in ((8, 2048), (512, 1024)):
        q = grid(nu, nv)
        assert binding.workspace_bytes(q) > 0
        binding.jit_check(q)                                                  # raises on a compile error
    for field in ("u", "wu", "v", "wv"):
        for bad in (float("nan"), float("inf")):
            a = np.array(getattr(base, field), dtype=float)
            a[3] = bad
            q = dataclasses.replace(base, **{field: a})
            with pytest.raises(binding.UgksError) as ei:
                binding.jit_check(q)
            assert ei.value.code == 1, (field, bad)
            keep, mesh, vg, gas, bcs = binding._structs(q)
            h = C.c_void_p()
            rc = libugks.ugks_init(C.byref(h), C.byref(mesh), C.byref(vg), C.byref(gas), C.byref(bcs), 0.8, C.c_void_p(256), 1 << 40, None)
            assert rc == 1 and b"finite" in libugks.ugks_last_error(None), (field, bad)


def test_generated_source_does_not_depend_on_the_locale():
    """the velocity nodes are written into the kernel source as hexadecimal literals built from their bits, so a host
    application running under a comma-radix LC_NUMERIC still compiles (printf("%a") would have written 0x1,8p+1)."""
    code = (
        "import locale, sys\n"
        "sys.path.insert(0, %r)\n"
        "ok = False\n"
        "for name in ('de_DE.UTF-8', 'de_DE.utf8', 'fr_FR.UTF-8', 'fr_FR.utf8', 'de_DE', 'fr_FR'):\n"
        "    try:\n"
        "        locale.setlocale(locale.LC_ALL, name); ok = True; break\n"
        "    except locale.Error:\n"
        "        pass\n"
        "if not ok or locale.localeconv()['decimal_point'] != ',':\n"
        "    print('NOLOCALE'); sys.exit(0)\n"
        "import workloads\n"
        "from paper_1810_08137_b200 import jit_check\n"
        "jit_check(workloads.channel_config('C1'))\n"
        "print('COMPILED')\n" % ROOT)
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    if "NOLOCALE" in r.stdout:
        pytest.skip("no comma-radix locale installed on this machine")
    assert "COMPILED" in r.stdout


def test_shipped_library_reads_no_environment_variable(libugks):
    """The experiment hooks (UGKS_JIT_DEFS pasted text into the kernel source) exist only in a -DUGKS_DEVELOPER build."""
    from paper_1810_08137_b200 import binding
    blob = open(binding.library_path(), "rb").read()
    for name in (b"UGKS_JIT_DEFS", b"UGKS_NSXM", b"UGKS_SLICE", b"UGKS_JIT_MAXREG", b"UGKS_JIT_DUMP", b"UGKS_DEBUG", b"UGKS_JIT_CHECK_TANGENTIAL"):
        assert name not in blob, name


def test_product_package_does_not_touch_the_oracle():
    """The product path may not import, link or read anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1810_08137_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in txt.lower() and "ugkso" not in txt, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_1810_08137_b200" not in txt or fn == "__init__.py" or "neither" in txt, fn
            assert "libugks.so" not in txt and "ugks_common" not in txt, fn


_RANK_SCRIPT = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import bench
rank, world, dist = bench.dist_setup(2, backend="gloo")
assert world == 2 and dist is not None
ms = bench.dist_max(dist, 10.0 + rank)            # max over ranks of the device time
pts = bench.dist_sum(dist, 100.0 * (rank + 1))    # replicas: points all ranks processed
dist.barrier()
if rank == 0:
    print(json.dumps({{"ms": ms, "pts": pts, "world": world}}))
dist.destroy_process_group()
"""


def test_bench_rank_plumbing_gloo_world_size_2(tmp_path):
    """bench.py --gpus N runs N replicas: value = sum of points / max-over-ranks time.  The helpers that do this are
    exercised with two gloo processes on CPU."""
    script = tmp_path / "rank.py"
    script.write_text(_RANK_SCRIPT.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
                          "127.0.0.1", "--master-port", "29517", str(script)], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1]
    r = json.loads(line)
    assert r == {"ms": 11.0, "pts": 300.0, "world": 2}


def test_reference_arm_prints_one_json_line_under_two_ranks():
    """--impl reference: rank 0 alone runs the oracle sample and prints the line; the other rank exits 0."""
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
                          "127.0.0.1", "--master-port", "29519", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "1", "--config", "C1"], env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    r = json.loads(lines[0])
    assert r["impl"] == "reference" and r["value"] > 0 and r["cpu_baseline"]["kind"] == "oracle"
    assert r["e2e"]["h2d_bytes_per_step"] == 0 and r["unit"] == "updates/s"
