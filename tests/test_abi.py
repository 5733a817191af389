"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/splx.h declares; the product path fails loudly without a CUDA device; the product
package never imports the oracle."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2606_18588_b200 import build
    return build.build()


def _declared():
    src = open(os.path.join(ROOT, "include", "splx.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(splx_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(libpath):
    names = _declared()
    assert len(names) >= 18 and "splx_project" in names and "splx_adam" in names
    L = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(L, n), n
    from paper_2606_18588_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_binding_mirrors_the_abi_names():
    from paper_2606_18588_b200 import binding
    for n in _declared():
        short = n[len("splx_"):]
        if short in ("create", "destroy", "last_error"):
            continue
        assert hasattr(binding.Context, short), short


def test_struct_sizes_match_the_header(libpath):
    from paper_2606_18588_b200 import binding as b
    assert ctypes.sizeof(b.Config) == 24
    assert ctypes.sizeof(b.CameraS) == 4 * (9 + 3 + 4) + 8 + 4
    assert ctypes.sizeof(b.GaussiansS) == 48 and ctypes.sizeof(b.ProjectedS) == 64
    assert ctypes.sizeof(b.BinningS) == 48 and ctypes.sizeof(b.PartialS) == 24


def test_iteration_structs_have_the_header_layout(tmp_path):
    """The ctypes mirrors of the splx_iteration structs against the C compiler's own layout of include/splx.h."""
    import subprocess
    from paper_2606_18588_b200 import binding as b
    src = tmp_path / "layout.c"
    src.write_text("""
#include <stdio.h>
#include <stddef.h>
#include "splx.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu ", sizeof(splx_frontset), sizeof(splx_trainset), sizeof(splx_bucket), sizeof(splx_adam_cfg),
         sizeof(splx_iter_opts), sizeof(splx_plan));
  printf("%zu %zu %zu %zu %zu %zu %zu\\n", offsetof(splx_trainset, part_offsets), offsetof(splx_trainset, bg),
         offsetof(splx_trainset, front), offsetof(splx_trainset, partials), offsetof(splx_trainset, loss_sum),
         offsetof(splx_trainset, touched), offsetof(splx_adam_cfg, m_soa));
  return 0;
}""")
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = [int(x) for x in subprocess.check_output([str(exe)]).split()]
    T, A = b.TrainsetS, b.AdamCfgS
    want = [ctypes.sizeof(b.FrontsetS), ctypes.sizeof(T), ctypes.sizeof(b.BucketS), ctypes.sizeof(A),
            ctypes.sizeof(b.IterOptsS), ctypes.sizeof(b.PlanS), T.part_offsets.offset, T.bg.offset, T.front.offset,
            T.partials.offset, T.loss_sum.offset, T.touched.offset, A.m_soa.offset]
    assert got == want


def test_cameras_with_a_bad_near_plane_are_rejected(libpath):
    """near_z <= 0 would admit z ~ 0 into 1/z and break the unsigned ordering of float_bits(depth); non-finite
    intrinsics likewise.  The host-only entry points can be called without a GPU."""
    import numpy as np
    from paper_2606_18588_b200 import binding as b, scenes
    lo = np.array([[-1, -1, 4]], np.float32); hi = np.array([[1, 1, 6]], np.float32)
    cam = scenes.Camera(np.eye(3, dtype=np.float32), np.zeros(3, np.float32), 50.0, 50.0, 16.0, 16.0, 32, 32)
    state, part = b.visible_regions(lo, hi, cam)
    assert part == 1
    for bad in (0.0, -0.5):
        cam.near_z = bad
        with pytest.raises(b.SplxError):
            b.visible_regions(lo, hi, cam)
        with pytest.raises(b.SplxError):
            b.visible_regions(lo, hi, cam, np.ones(1, np.float32))


def test_no_cpu_fallback_without_a_device(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2606_18588_b200 import binding
    with pytest.raises(binding.SplxError) as e:
        binding.Context(0)
    assert "no CPU fallback" in str(e.value) or "no CUDA device" in str(e.value)
    # and straight through the C ABI
    L = binding.lib()
    h = ctypes.c_void_p()
    rc = L.splx_create(ctypes.byref(h), 0, None, None)
    assert rc == binding.ERR_CUDA and not h.value
    assert b"no CUDA device" in L.splx_last_error(None)


def test_product_package_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_18588_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "liboracle" not in txt and "splx_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2606_18588_b200\b", txt, flags=re.M), f
            assert "libsplx" not in txt
