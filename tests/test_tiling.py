"""Host logic of the resident kernel: tile / box geometry (paper_1507_08549_b200/csrc/tiling.h), brute-forced on CPU.

tiling.h is plain C++ shared by the host planner and the device code.  The kernel is only correct if, for every
tile, the fixed-size box contains the owned interval widened by the 2m-cell dependency margin of m red-black sweeps
(DESIGN.md §6).  This file compiles the header with g++ and checks that property, and the partition property, for
every (n, B, h, q) the planner can meet.
"""
import ctypes as C
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HDR = os.path.join(ROOT, "paper_1507_08549_b200", "csrc", "tiling.h")

SRC = r'''
#include "%s"
extern "C" {
int t_plan_axis(int n, int B, int h, int q, int* nt, int* own) { return snp::plan_axis(n, B, h, q, nt, own) ? 1 : 0; }
int t_box_origin(int x0, int h, int q, int B, int n) { return snp::box_origin(x0, h, q, B, n); }
int t_box_covers(int t, int own, int h, int q, int B, int n) { return snp::box_covers(t, own, h, q, B, n) ? 1 : 0; }
}
'''


@pytest.fixture(scope="module")
def til(tmp_path_factory):
    d = tmp_path_factory.mktemp("tiling")
    src = d / "t.cpp"
    src.write_text(SRC % HDR)
    so = d / "libt.so"
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-fPIC", "-shared", "-o", str(so), str(src)])
    lib = C.CDLL(str(so))
    ip = C.POINTER(C.c_int)
    lib.t_plan_axis.argtypes = [C.c_int] * 4 + [ip, ip]
    lib.t_box_origin.argtypes = [C.c_int] * 5
    lib.t_box_covers.argtypes = [C.c_int] * 6
    return lib


def plan(lib, n, B, h, q):
    nt, own = C.c_int(0), C.c_int(0)
    ok = lib.t_plan_axis(n, B, h, q, C.byref(nt), C.byref(own))
    return (nt.value, own.value) if ok else None


# (alignment q, box extents B) the kernel shapes use: r axis q = 4, z axis q = H in {2, 4, 8}
AXES = [(4, (32, 64, 128)), (2, (32,)), (4, (32,)), (8, (64, 112))]


@pytest.mark.parametrize("q,boxes", AXES)
def test_every_plan_partitions_the_axis_and_every_box_covers_its_margin(til, q, boxes):
    checked = 0
    for B in boxes:
        for m in range(1, 9):
            h = 2 * m
            for n in list(range(q, 6 * B + q, q)) + [512, 1024, 2048, 4096]:
                if n % q:
                    continue
                p = plan(til, n, B, h, q)
                if p is None:
                    continue
                nt, own = p
                assert own % q == 0 and own >= q
                assert (nt - 1) * own < n <= nt * own, (n, B, h, q, nt, own)      # tiles tile [0, n), none empty
                for t in range(nt):
                    x0, x1 = t * own, min(n, (t + 1) * own)
                    o = til.t_box_origin(x0, h, q, B, n)
                    assert o % q == 0 and 0 <= o and o + B <= n
                    assert o <= max(x0 - h, 0) and o + B >= min(x1 + h, n), (n, B, h, q, t, o)
                    assert til.t_box_covers(t, own, h, q, B, n) == 1
                    # the kernel gates its halo reload on the flags of tiles [o/own, (o+B-1)/own]: every tile that
                    # owns a cell of the box must be in that range
                    lo_t, hi_t = o // own, (o + B - 1) // own
                    assert lo_t <= t <= hi_t and hi_t < nt
                    checked += 1
    assert checked > 1000


def test_plan_rejects_what_cannot_fit(til):
    assert plan(til, 30, 32, 2, 4) is None            # grid smaller than one box
    assert plan(til, 34, 32, 2, 4) is None            # not a multiple of the alignment
    assert plan(til, 64, 32, 16, 4) is None           # margins eat the whole box
    assert plan(til, 32, 32, 16, 4) == (1, 32)        # box == grid: one tile, no margins needed
    nt, own = plan(til, 512, 128, 8, 4)
    assert nt * own >= 512 and own <= 128 - 2 * 8


def test_box_covers_detects_a_bad_tiling(til):
    # owned 120 of a 128-box with margin 8 on both sides cannot be covered in the middle of a 512 axis
    assert til.t_box_covers(1, 120, 8, 4, 128, 512) == 0
    assert til.t_box_covers(1, 112, 8, 4, 128, 512) == 1
