"""GPU: the -DART_DEBUG build of the library validates device-side contents and traps ("Errors": release
builds do not look at page ids or list entries; a debug build traps).  Every case runs in its own process: a trap ends
the CUDA context of the process it happens in."""
import os
import subprocess
import sys
import textwrap

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PKG = os.path.join(ROOT, "paper_2606_00024_b200")
DEBUG_LIB = os.path.join(PKG, "libart_decode_debug.so")


@pytest.fixture(scope="module")
def debug_lib():
    env = dict(os.environ, ART_BUILD_TAG="debug", ART_NVCC_FLAGS="-DART_DEBUG")
    subprocess.run([sys.executable, os.path.join(PKG, "build.py")], check=True, env=env, cwd=ROOT)
    assert os.path.exists(DEBUG_LIB)
    return DEBUG_LIB


CHILD = textwrap.dedent("""
    import ctypes, sys
    sys.path.insert(0, {root!r}); sys.path.insert(0, {root!r} + "/tests")
    import torch
    import paper_2606_00024_b200 as art
    from workloads import generators as gen
    lib = art.load_library()
    assert hasattr(lib, "art_debug_last_violation"), "not the debug build"
    lib.art_debug_last_violation.restype = ctypes.c_ulonglong
    w = gen.config({index}, scale=1 / 16, batch=2).to("cuda")
    {corrupt}
    try:
        out, stop, _ = art.run_workload(w, art={art_on})
        torch.cuda.synchronize()
    except Exception as e:
        val = ctypes.c_ulonglong(0)
        v = lib.art_debug_last_violation(ctypes.byref(val))
        print("TRAPPED code=%d b=%d g=%d index=%d value=%d" % (v >> 48, (v >> 32) & 0xffff, (v >> 24) & 0xff, v & 0xffffff, val.value))
        sys.exit(3)
    print("OK stop", stop.flatten()[:4].tolist())
""")


def run_child(lib, index, corrupt, art_on=True):
    code = CHILD.format(root=ROOT, index=index, corrupt=corrupt, art_on=art_on)
    env = dict(os.environ, ART_LIB_PATH=lib)
    return subprocess.run([sys.executable, "-c", code], env=env, cwd=ROOT, capture_output=True, text=True, timeout=240)


def test_clean_inputs_pass_under_the_debug_build(debug_lib):
    for index, art_on in ((1, True), (1, False), (2, True), (3, False)):
        r = run_child(debug_lib, index, "pass", art_on)
        assert r.returncode == 0 and "OK stop" in r.stdout, (index, art_on, r.stdout[-400:], r.stderr[-400:])


def test_page_id_out_of_range_traps(debug_lib):
    r = run_child(debug_lib, 1, "w.block_table[1, 3] = w.k_cache.shape[0]")
    assert r.returncode == 3 and "TRAPPED code=5 b=1" in r.stdout and "index=3" in r.stdout, (r.stdout[-400:], r.stderr[-400:])
    r = run_child(debug_lib, 1, "w.block_table[0, 0] = -1", art_on=False)
    assert r.returncode == 3 and "TRAPPED code=5 b=0" in r.stdout, (r.stdout[-400:], r.stderr[-400:])


def test_bad_list_entries_trap(debug_lib):
    r = run_child(debug_lib, 2, "w.eligible_blocks[1, 2, 5] = w.eligible_blocks[1, 2, 1]")           # a repeated entry
    assert r.returncode == 3 and "TRAPPED code=4 b=1 g=2 index=5" in r.stdout, (r.stdout[-400:], r.stderr[-400:])
    r = run_child(debug_lib, 2, "w.eligible_blocks[0, 1, 2] = w.block_table.shape[1]")               # beyond the table
    assert r.returncode == 3 and "TRAPPED code=3 b=0 g=1 index=2" in r.stdout, (r.stdout[-400:], r.stderr[-400:])
    r = run_child(debug_lib, 2, "w.eligible_counts[1, 0] = w.eligible_blocks.shape[2] + 1")          # count beyond the row
    assert r.returncode == 3 and "TRAPPED code=2 b=1 g=0" in r.stdout, (r.stdout[-400:], r.stderr[-400:])


def test_sequence_length_beyond_the_table_traps(debug_lib):
    r = run_child(debug_lib, 1, "w.seq_lens[0] = w.block_table.shape[1] * 64 + 1", art_on=False)
    assert r.returncode == 3 and "TRAPPED code=1 b=0" in r.stdout, (r.stdout[-400:], r.stderr[-400:])
