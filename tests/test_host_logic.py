"""-m "not gpu": the C-ABI library builds for sm_100a, loads without a GPU and exports every symbol the header
declares; host-only entry points; bench.py's max-over-ranks reduction on 2 gloo ranks."""
import ctypes as C
import os
import re
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def fp():
    import paper_2510_00518_b200 as fp
    fp.build_library()
    fp.load_library()
    return fp


def test_library_exports_every_declared_symbol(fp):
    header = (ROOT / "include" / "fourphonon.h").read_text()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(fp_[a-z0-9_]+)\s*\(", header))
    assert declared == set(fp.EXPORTED_SYMBOLS), declared ^ set(fp.EXPORTED_SYMBOLS)
    lib = C.CDLL(str(fp.library_path()))
    for sym in declared:
        assert hasattr(lib, sym), sym
    out = subprocess.run(["nm", "-D", "--defined-only", str(fp.library_path())], capture_output=True, text=True).stdout
    for sym in declared:
        assert re.search(rf"\bT {sym}\b", out), f"{sym} is not an exported text symbol"


def test_library_targets_sm_100a(fp):
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", str(fp.library_path())], capture_output=True,
                         text=True).stdout
    assert "sm_100a" in out


def test_constants_against_codata_closed_forms(fp):
    """tests/golden/constants.txt: SURVEY.md §8(c) 'Constants' (CODATA 2018 exact/recommended values)."""
    c = fp.fp_constants()
    hbar, kb, qe, amu = 1.054571817e-34, 1.380649e-23, 1.602176634e-19, 1.66053906660e-27
    assert abs(c["hbar_over_kb"] - hbar / kb * 1e12) < 1e-12 * c["hbar_over_kb"]
    c3 = np.pi * hbar / 4 * (qe / 1e-30) ** 2 / amu ** 3 / (1e12) ** 4 / 1e12
    c4 = np.pi * hbar ** 2 / 8 * (qe / 1e-40) ** 2 / amu ** 4 / (1e12) ** 5 / 1e12
    assert abs(c["C3"] - c3) < 1e-12 * c3 and abs(c["C4"] - c4) < 1e-12 * c4
    assert abs(c["C3"] - 4.643436782e8) < 1e-9 * c3 and abs(c["C4"] - 1.474472255e9) < 1e-9 * c4
    assert abs(c["Ckappa"] - 8.055064808) < 1e-9 * 8.055064808


def test_workspace_bytes_host_only(fp):
    from paper_2510_00518_b200.binding import _Crystal
    lib = fp.load_library()
    cr = _Crystal()
    cr.natoms = 2
    mesh = (C.c_int32 * 3)(16, 16, 16)
    small = lib.fp_workspace_bytes(C.byref(cr), mesh, None, None, 1 << 20)
    big = lib.fp_workspace_bytes(C.byref(cr), mesh, None, None, 1 << 30)
    assert 0 < small < big and big >= (1 << 30)
    assert small >= 24576 * (32 + 8 + 6 * 16)                              # resident mode tables
    bad = (C.c_int32 * 3)(16, 0, 16)
    assert lib.fp_workspace_bytes(C.byref(cr), bad, None, None, 1 << 20) == 0
    cr.natoms = 0
    assert lib.fp_workspace_bytes(C.byref(cr), mesh, None, None, 1 << 20) == 0


def test_setup_rejects_bad_arguments_without_touching_the_gpu(fp):
    """Argument errors are detected on the host before any CUDA call (FP_EINVAL, message set)."""
    from paper_2510_00518_b200.binding import _Crystal, _Broadening
    lib = fp.load_library()
    cr = _Crystal(); cr.natoms = 1
    cr.lattvec = (C.c_double * 9)(3, 0, 0, 0, 3, 0, 0, 0, 3)
    mesh = (C.c_int32 * 3)(2, 2, 2)
    br = _Broadening(1.0, 2.0, 0.0)
    ctx = C.c_void_p(None)
    dummy = (C.c_double * 1024)()
    ws = C.c_void_p(256)
    rc = lib.fp_setup(C.byref(cr), dummy, dummy, dummy, dummy, 0, None, None, mesh, -5.0, C.byref(br), ws, 1 << 20, None,
                      C.byref(ctx))
    assert rc == fp.FP_EINVAL and b"T" in lib.fp_last_error(None)
    br2 = _Broadening(0.0, 2.0, 0.0)
    rc = lib.fp_setup(C.byref(cr), dummy, dummy, dummy, dummy, 0, None, None, mesh, 300.0, C.byref(br2), ws, 1 << 20, None,
                      C.byref(ctx))
    assert rc == fp.FP_EINVAL
    rc = lib.fp_setup(C.byref(cr), dummy, dummy, dummy, dummy, 0, None, None, mesh, 300.0, C.byref(br), C.c_void_p(257),
                      1 << 20, None, C.byref(ctx))
    assert rc == fp.FP_EINVAL and not ctx.value


def test_missing_library_fails_loudly(fp, monkeypatch, tmp_path):
    import paper_2510_00518_b200.binding as b
    monkeypatch.setattr(b, "_lib", None)
    monkeypatch.setattr(b, "_LIB", tmp_path / "nope.so")
    with pytest.raises(b.FourPhononError):
        b.load_library()


def test_product_path_never_imports_the_oracle():
    files = list((ROOT / "paper_2510_00518_b200").rglob("*.py")) + list((ROOT / "paper_2510_00518_b200").rglob("*.cu*")) + \
        list((ROOT / "include").glob("*.h")) + list((ROOT / "fp_inputs").glob("*.py"))
    assert len(files) >= 6
    for p in files:
        txt = p.read_text()
        assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f"{p} imports the oracle"
        assert "fp_oracle" not in txt and not re.search(r"#include\s+[\"<][^\n]*oracle", txt), f"{p} links the oracle"


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo", rank=int(sys.argv[1]), world_size=2, init_method="tcp://127.0.0.1:{port}")
r = int(sys.argv[1])
ms, units = bench.reduce_over_ranks(10.0 + 5.0 * r, 100.0 * (r + 1), dist)
assert ms == 15.0 and units == 300.0, (ms, units)
dist.destroy_process_group()
print("ok")
"""


def test_reduce_over_ranks_gloo_world2(tmp_path):
    port = 29000 + os.getpid() % 2000
    script = tmp_path / "w.py"
    script.write_text(_WORKER.format(root=str(ROOT), port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                              text=True) for r in range(2)]
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0 and "ok" in out, err


def test_reference_arm_nonzero_rank_exits_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2"], env=env,
                       capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
