"""The C-ABI library builds, loads, and exports every function include/*.h declares (no GPU needed)."""
import ctypes
import glob
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    names = []
    for h in glob.glob(os.path.join(ROOT, "include", "*.h")):
        src = re.sub(r"/\*.*?\*/", "", open(h).read(), flags=re.S)
        names += re.findall(r"^\s*(?:int32_t|const char\*)\s+(db_\w+)\s*\(", src, flags=re.M)
    return sorted(set(names))


def test_header_declares_the_north_star_calls():
    d = _declared()
    for f in ("db_create", "db_step", "db_read_spikes", "db_read_state", "db_region_rates"):
        assert f in d


def test_library_exports_every_declared_symbol():
    import paper_2211_15963_b200 as db
    lib = ctypes.CDLL(db.build())
    for f in _declared():
        assert hasattr(lib, f), f
    assert sorted(db.binding.EXPORTS) == _declared()


def test_struct_sizes_match_the_header():
    # compile a tiny C program against the header and compare sizeof with the ctypes mirrors
    import subprocess, tempfile
    import paper_2211_15963_b200.binding as b
    code = r'''
#include <stdio.h>
#include "db_b200.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu %zu %zu\n", sizeof(db_type_params), sizeof(db_sim_params), sizeof(db_runtime),
         sizeof(db_network_spec), sizeof(db_csr_view), sizeof(db_csr_host), sizeof(db_counters), sizeof(db_phase_times));
  return 0; }'''
    with tempfile.TemporaryDirectory() as td:
        src = os.path.join(td, "s.c")
        open(src, "w").write(code)
        exe = os.path.join(td, "s")
        subprocess.check_call(["gcc", "-std=c11", "-I", os.path.join(ROOT, "include"), src, "-o", exe])
        got = [int(x) for x in subprocess.check_output([exe]).split()]
    want = [ctypes.sizeof(x) for x in (b.TypeParams, b.SimParams, b.Runtime, b.NetworkSpec, b.CsrView, b.CsrHost,
                                       b.Counters, b.PhaseTimes)]
    assert got == want


def test_create_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import db_inputs
    import paper_2211_15963_b200 as db
    with pytest.raises(RuntimeError):
        db.Sim.db_create_from_csr(db_inputs.sim_params(), db_inputs.random_csr(64, 5, 1))
    # and the raw C call reports DB_ECUDA rather than falling back
    L = db.load()
    sp = db.binding.SimParams()
    db.binding._fill_sim_params(sp, db_inputs.sim_params(), 1, 0, 0, 0)
    import numpy as np
    net = db_inputs.random_csr(64, 5, 1)
    keep = [np.ascontiguousarray(net["region_start"], np.int64), net["ntype"], net["row_ptr"], net["tgt"], net["w"],
            net["delay"], net["rec"]]
    v = db.binding.CsrView(64, int(net["E"]), 1, *[a.ctypes.data_as(ctypes.c_void_p) for a in keep], 0)
    h = ctypes.c_void_p()
    rc = L.db_create_from_csr(ctypes.byref(sp), ctypes.byref(v), None, ctypes.byref(h))
    assert rc == db.binding.DB_ECUDA and not h
    assert b"CUDA" in L.db_last_error(None)


def test_create_from_csr_rejects_bad_sizes_before_touching_the_arrays():
    # N, E and n_regions are checked before row_ptr[N] or delay[0..E) is read (no device needed: the checks come first)
    import numpy as np
    import db_inputs
    import paper_2211_15963_b200 as db
    L = db.load()
    sp = db.binding.SimParams()
    db.binding._fill_sim_params(sp, db_inputs.sim_params(), 1, 0, 0, 0)
    net = db_inputs.random_csr(64, 5, 1)
    keep = [np.ascontiguousarray(net["region_start"], np.int64), net["ntype"], net["row_ptr"], net["tgt"], net["w"],
            net["delay"], net["rec"]]
    ptrs = [a.ctypes.data_as(ctypes.c_void_p) for a in keep]
    for N, E, R in ((-1, 10, 1), (0, 0, 1), (1 << 30, 10, 1), (64, -3, 1), (64, int(net["E"]), 0), (64, int(net["E"]), 70000)):
        v = db.binding.CsrView(N, E, R, *ptrs, 0, 0, 0)
        h = ctypes.c_void_p()
        rc = L.db_create_from_csr(ctypes.byref(sp), ctypes.byref(v), None, ctypes.byref(h))
        assert rc == db.binding.DB_EINVAL and not h, (N, E, R, rc)
    v = db.binding.CsrView(64, int(net["E"]), 1, None, *ptrs[1:], 0, 0, 0)          # a missing array
    h = ctypes.c_void_p()
    assert L.db_create_from_csr(ctypes.byref(sp), ctypes.byref(v), None, ctypes.byref(h)) == db.binding.DB_EINVAL
