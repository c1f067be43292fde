"""-m "not gpu": the C-ABI library builds, loads without a GPU and exports every symbol include/mcx.h declares;
host-only entry points (workspace size, argument validation) behave as documented."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2410_08747_b200 import binding
    binding.lib()
    return binding


def declared_functions():
    text = open(os.path.join(ROOT, "include", "mcx.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mcx_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(B):
    names = declared_functions()
    assert len(names) >= 12
    L = C.CDLL(os.path.join(ROOT, "paper_2410_08747_b200", "libmcx_b200.so"))
    for n in names:
        assert hasattr(L, n), n
    assert sorted(B.EXPORTS) == names


def test_struct_sizes_match_the_header(B):
    # compile a tiny C program against include/mcx.h and compare sizeof with the ctypes mirrors
    import subprocess, tempfile
    src = r'''
#include <stdio.h>
#include "mcx.h"
int main(void) { printf("%zu %zu %zu %zu %zu\n", sizeof(mcx_component), sizeof(mcx_solid), sizeof(mcx_material),
                        sizeof(mcx_ray_fate), sizeof(mcx_pose)); return 0; }
'''
    with tempfile.TemporaryDirectory() as d:
        p = os.path.join(d, "s.c")
        open(p, "w").write(src)
        exe = os.path.join(d, "s")
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", exe, p])
        sizes = [int(x) for x in subprocess.check_output([exe]).split()]
    assert sizes == [C.sizeof(B.McxComponent), C.sizeof(B.McxSolid), C.sizeof(B.McxMaterial), B.FATE_DTYPE.itemsize,
                     C.sizeof(B.McxPose)]


def _marshal(B, inst):
    keep = []
    comps, mats = B.marshal(inst, keep, lambda ids: 0x1000)   # fake device pointer: the size query never reads it
    return comps, mats, keep


def test_workspace_size_counts_the_tallies(B, W):
    L = B.lib()
    for k, kw in ((0, {}), (1, {"small": True}), (2, {"small": True}), (3, {"small": True}), (4, {"small": True})):
        inst = W.config(k, **kw)
        comps, mats, keep = _marshal(B, inst)
        n = C.c_size_t()
        assert L.mcx_instrument_workspace_size(comps, len(inst["components"]), mats, len(inst["materials"]), C.byref(n)) == 0
        bins = sum(W.n_bins(d) for d in W.detectors_of(inst))
        assert n.value >= 32 * bins and n.value % 256 == 0
        if k == 4:
            assert n.value >= 32 * bins + inst["components"][1]["ids"].size


def test_workspace_size_counts_the_staged_trace(B, W):
    # a chain of slits, voxel volumes and detectors whose volume scatters is traced in stages (include/mcx.h, mcx_tuning
    # staged_walk): its workspace holds the pool of 2^22 ray records of 80 bytes and, for a volume of at most 16
    # materials, the one-byte cells; the same chain without scattering, or with a solids group in it, holds neither
    L = B.lib()
    def size(inst):
        comps, mats, keep = _marshal(B, inst)
        n = C.c_size_t()
        assert L.mcx_instrument_workspace_size(comps, len(inst["components"]), mats, len(inst["materials"]), C.byref(n)) == 0
        return n.value
    pool = 80 << 22
    plain, scat = W.config4(small=True), W.config4(small=True, scatter_order=2)
    cells = plain["components"][1]["ids"].size
    assert size(scat) - size(plain) >= pool + cells and size(scat) - size(plain) < pool + 4 * cells + (1 << 20)
    many = W.config4(small=True, scatter_order=2)
    many["materials"] = list(many["materials"]) + [many["materials"][1]] * 4     # 20 materials: no one-byte cells
    assert pool <= size(many) - size(plain) < size(scat) - size(plain)
    mixed = W.config4(small=True, scatter_order=2)
    mixed["components"] = mixed["components"][:2] + [W.solids([W.solid_sphere(0.006, 1, 0, T=(0.0, 0.0, 0.9))])] + mixed["components"][2:]
    assert size(mixed) - size(plain) < pool


def test_argument_errors_are_reported_synchronously(B, W):
    L = B.lib()
    inst = W.config0()
    comps, mats, keep = _marshal(B, inst)
    n = C.c_size_t()
    assert L.mcx_instrument_workspace_size(comps, len(inst["components"]), mats, 2, None) == 1
    assert b"bytes_out" in L.mcx_last_error()
    comps[0].kind = 1                                  # chain no longer starts with a source
    assert L.mcx_instrument_workspace_size(comps, 4, mats, 2, C.byref(n)) == 1
    assert b"source" in L.mcx_last_error()
    comps[0].kind = 0
    assert L.mcx_instrument_workspace_size(comps, 17, mats, 2, C.byref(n)) == 2   # MCX_ERR_UNSUPPORTED
    h = C.c_void_p()
    assert L.mcx_instrument_create(comps, 4, mats, 2, None, 0, None, C.byref(h)) == 4   # MCX_ERR_WORKSPACE
    assert L.mcx_instrument_create(comps, 4, mats, 2, 0x1001, 1 << 30, None, C.byref(h)) == 4  # misaligned
    assert L.mcx_trace(None, 10, 1, None) == 1
    assert L.mcx_launch_count(None) == 0
