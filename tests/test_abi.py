"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, exports
every symbol include/afm.h declares, validates arguments before touching the
device, and fails loudly (no CPU fallback) when no GPU is present."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

from paper_1109_0334_b200 import afm, build, workloads as wlm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "afm.h")


@pytest.fixture(scope="module")
def lib():
    build.build()
    return afm.lib()


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(afm_[a-z0-9_]+)\s*\(", src)))


def test_header_functions_are_all_exported(lib):
    names = _declared_functions()
    assert len(names) >= 10
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(afm.SYMBOLS) == names


def test_struct_layouts_match_the_header(tmp_path):
    """Size of every POD of afm.h and offset of every field, as the C compiler lays
    them out, against the ctypes mirrors of the binding."""
    pods = (("afm_cfg", afm.Cfg), ("afm_bounds", afm.Bounds), ("afm_swarm_cfg", afm.SwarmCfg),
            ("afm_beam_cfg", afm.BeamCfg))
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "afm.h"', 'int main(){']
    want = []
    for cname, cls in pods:
        lines.append('printf("%%zu\\n", sizeof(%s));' % cname)
        want.append(C.sizeof(cls))
        for fname, _ in cls._fields_:
            lines.append('printf("%%zu\\n", offsetof(%s, %s));' % (cname, fname))
            want.append(getattr(cls, fname).offset)
    lines.append('return 0;}')
    src, exe = tmp_path / "abi_layout.c", tmp_path / "abi_layout"
    src.write_text("\n".join(lines))
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = [int(x) for x in subprocess.check_output([str(exe)]).split()]
    assert got == want


def test_library_is_sm100a_and_uses_bulk_async_copy():
    out = subprocess.check_output(["cuobjdump", "-lelf", afm.LIB_PATH]).decode()
    assert "sm_100a" in out
    sass = subprocess.check_output(["cuobjdump", "-sass", afm.LIB_PATH]).decode()
    assert "UBLKCP" in sass          # cp.async.bulk: the TMA-staged time tiles
    assert "SYNCS" in sass           # mbarrier
    assert "MUFU.RCP64H" in sass and "DFMA" in sass


def test_validation_happens_before_the_device_is_touched(lib):
    wl = wlm.config(0)
    for field, val in (("n_params", 3), ("steps_per_cycle", 0), ("n_skip_cycles", 20),
                       ("law", 7), ("n_traces", 0), ("k", -1.0), ("precision", 5)):
        cfg = afm.cfg_from(wl, **{field: val})
        rc = lib.afm_forward_batch(C.c_void_p(16), 4, C.c_void_p(16), C.byref(cfg), None,
                                   C.c_void_p(16), None)
        assert rc == afm.EINVAL, field
        assert afm.afm_last_error()
    cfg = afm.cfg_from(wl)
    assert lib.afm_forward_batch(None, 4, C.c_void_p(16), C.byref(cfg), None,
                                 C.c_void_p(16), None) == afm.EINVAL
    assert lib.afm_forward_batch(C.c_void_p(16), 0, C.c_void_p(16), C.byref(cfg), None,
                                 C.c_void_p(16), None) == afm.EINVAL
    cfg3 = afm.cfg_from(wl, n_traces=3)
    assert lib.afm_forward_batch(C.c_void_p(16), 4, C.c_void_p(16), C.byref(cfg3), None,
                                 C.c_void_p(16), None) == afm.EINVAL
    b = afm.bounds_from(wl)
    b.lo[0] = 5.0
    b.hi[0] = 1.0
    th = np.zeros(2)
    rc = lib.afm_pso_invert(C.byref(b), C.byref(afm.swarm_from(wl)), 0, C.c_void_p(16),
                            C.byref(cfg), th.ctypes.data, th.ctypes.data, None, None, None,
                            None)
    assert rc == afm.EINVAL
    assert afm.afm_set_option("block", 0) is None
    with pytest.raises(afm.AfmError):
        afm.afm_set_option("block", 48)
    with pytest.raises(afm.AfmError):
        afm.afm_set_option("nonsense", 1)


def test_no_cpu_fallback_without_a_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    wl = wlm.config(0)
    cfg = afm.cfg_from(wl)
    th = np.zeros(2)
    rc = lib.afm_forward_batch_host(th.ctypes.data, 1, np.zeros(wl["n_window"]).ctypes.data,
                                    C.byref(cfg), None, th.ctypes.data, None)
    assert rc in (afm.ECUDA, afm.EUNSUPPORTED)
    assert "CUDA" in afm.afm_last_error() or "device" in afm.afm_last_error()


def test_product_package_never_imports_the_oracle():
    """The product path shares nothing with oracle/: no import, include, dlopen."""
    pkg = os.path.join(ROOT, "paper_1109_0334_b200")
    pat = re.compile(r"import\s+oracle|from\s+oracle|oracle[./]|afm_oracle|orc_[a-z]")
    for top in (pkg, os.path.join(ROOT, "include")):
        for dirpath, _, files in os.walk(top):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h")):
                    text = open(os.path.join(dirpath, f)).read()
                    assert not pat.search(text), (f, pat.search(text).group(0))


def test_queue_status_is_ok_before_any_queue_kernel_has_run(lib):
    """afm_queue_status has nothing to wait for, and makes no CUDA call, until a
    segment-queue kernel has been launched (this runs on a box with no GPU)."""
    assert lib.afm_queue_status(None) == afm.OK


def test_pso_step_host_validates_like_pso_step(lib):
    """The host-buffer step checks bounds and iteration up front (it used to leave
    that to the device-buffer call, after staging)."""
    w0 = wlm.config(0)
    b, sw = afm.bounds_from(w0), afm.swarm_from(w0)
    p16 = C.c_void_p(16)
    args = lambda bb, it: (C.byref(bb), C.byref(sw), 2, 1, 0, it, 1, p16, p16, p16, p16,
                           p16, p16, p16, None)
    assert lib.afm_pso_step_host(*args(b, -1)) == afm.EINVAL
    bad = afm.bounds_from(w0)
    bad.lo[0], bad.hi[0] = 2.0, 1.0
    assert lib.afm_pso_step_host(*args(bad, 0)) == afm.EINVAL
    assert lib.afm_pso_step(*args(bad, 0)) == afm.EINVAL


def test_new_entry_points_validate_before_touching_the_device(lib):
    """Beam model, sharded swarm, probes, options: bad arguments are AFM_EINVAL
    without any CUDA call (this runs on a box with no GPU)."""
    wl = wlm.beam_workload()
    p16 = C.c_void_p(16)
    for field, val in (("n_modes", 3), ("n_points", 500), ("n_points", 1), ("Q", 0.0),
                       ("n_params", 3), ("law", 9), ("n_skip_cycles", 80), ("n_traces", 0),
                       ("L", -1.0), ("A_ref", 0.0)):
        cfg = afm.beam_cfg_from(wl, **{field: val})
        rc = lib.afm_beam_forward_batch(p16, 4, p16, C.byref(cfg), None, p16, None)
        assert rc == afm.EINVAL, (field, val)
        assert lib.afm_beam_modes(C.byref(cfg), None, None, None, None, None, None) == afm.EINVAL
        assert lib.afm_beam_trajectory(p16, C.byref(cfg), None, None, None) == afm.EINVAL
    cfg = afm.beam_cfg_from(wl)
    assert lib.afm_beam_forward_batch(p16, 3, p16, C.byref(afm.beam_cfg_from(wl, n_traces=2)),
                                      None, p16, None) == afm.EINVAL
    assert lib.afm_beam_forward_batch(None, 4, p16, C.byref(cfg), None, p16, None) == afm.EINVAL
    w0 = wlm.config(0)
    b, sw, c0 = afm.bounds_from(w0), afm.swarm_from(w0), afm.cfg_from(w0)
    assert lib.afm_pso_shard_init(C.byref(b), C.byref(sw), 2, 1, 0, -1, p16, p16, p16, p16,
                                  p16, p16, None) == afm.EINVAL
    assert lib.afm_pso_shard_eval(C.byref(b), C.byref(sw), p16, C.byref(c0), -5, p16, p16,
                                  p16, p16, p16, None) == afm.EINVAL
    def shard_move(n_ranks=1, rank=0, total=64, swarm=sw, pbestJ=p16):
        return lib.afm_pso_shard_move(C.byref(b), C.byref(swarm), 2, 1, 0, 0, 1, 0, p16,
                                      n_ranks, rank, total, p16, p16, p16, pbestJ, p16, p16,
                                      None, None, None)
    assert shard_move(n_ranks=0) == afm.EINVAL
    assert shard_move(n_ranks=2, rank=2) == afm.EINVAL
    assert shard_move(total=10) == afm.EINVAL          # smaller than the shard itself
    ring = afm.swarm_from(w0, topology=1)
    assert shard_move(swarm=ring, pbestJ=None) == afm.EINVAL
    chunked = afm.swarm_from(w0, async_chunk=8)
    assert shard_move(swarm=chunked) == afm.EUNSUPPORTED
    assert lib.afm_pso_shard_eval(C.byref(b), C.byref(chunked), p16, C.byref(c0), 0, p16, p16,
                                  p16, p16, p16, None) == afm.EUNSUPPORTED
    assert lib.afm_pso_step(C.byref(b), C.byref(chunked), 2, 1, 0, 0, 1, p16, p16, p16, p16,
                            p16, p16, p16, None) == afm.EUNSUPPORTED
    bad = afm.swarm_from(w0, async_chunk=-1)
    assert lib.afm_pso_step(C.byref(b), C.byref(bad), 2, 1, 0, 0, 1, p16, p16, p16, p16,
                            p16, p16, p16, None) == afm.EINVAL
    out = C.c_double(0.0)
    assert lib.afm_fma_peak(7, 0.1, C.byref(out), None) == afm.EINVAL
    assert lib.afm_fma_peak(0, 100.0, C.byref(out), None) == afm.EINVAL
    ms, n = (C.c_double * 4)(), C.c_int32(0)
    assert lib.afm_kernel_times(None, 4, C.byref(n)) == afm.EINVAL
    assert lib.afm_kernel_times(ms, 4, C.byref(n)) == afm.OK and n.value == 0
    z = np.zeros(8)
    assert lib.afm_pso_step_host(C.byref(b), C.byref(sw), 9, 1, 0, 0, 1, z.ctypes.data,
                                 z.ctypes.data, z.ctypes.data, z.ctypes.data, z.ctypes.data,
                                 z.ctypes.data, z.ctypes.data, None) == afm.EINVAL
    assert lib.afm_pso_step_host(C.byref(b), C.byref(sw), 2, 1, 0, 0, 1, None, z.ctypes.data,
                                 z.ctypes.data, z.ctypes.data, z.ctypes.data, z.ctypes.data,
                                 z.ctypes.data, None) == afm.EINVAL
    for name, bad in (("form", 3), ("lanes", 3), ("pack", 5), ("ppt", 4), ("tile", -1),
                      ("queue", 3), ("segs", 5000), ("workers", 9), ("boost", 65), ("boost2", 2),
                      ("kernel_events", 2)):
        with pytest.raises(afm.AfmError):
            afm.afm_set_option(name, bad)
        assert afm.afm_set_option(name, 0) is None
