"""`-m "not gpu"`: the C-ABI library builds, loads and exports every symbol include/farm.h declares; host-side
argument validation works without a GPU; the product path fails loudly (no CPU fallback)."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_15476_b200 import build, binding
    build.build()
    return binding.load_library()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "farm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(farm_[a-z_]+)\s*\(", hdr))
    assert len(names) >= 16
    from paper_2606_15476_b200 import binding
    assert names == set(binding.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n


def test_struct_layouts_match_header():
    from paper_2606_15476_b200 import binding
    assert binding.OBJECT_DTYPE.itemsize == 72 and binding.OBJECT_DTYPE.fields["n_points"][1] == 64
    assert binding.STATS_DTYPE.itemsize == 48 and binding.TOTALS_DTYPE.itemsize == 48


def test_host_side_validation_without_gpu(lib):
    from paper_2606_15476_b200 import FarmError, FarmMap
    with pytest.raises(FarmError):
        FarmMap(0.0, 64, 0.5, 0.5, 0.5, H=8, W=8)            # voxel_size must be > 0
    with pytest.raises(FarmError):
        FarmMap(0.05, 0, 0.5, 0.5, 0.5, H=8, W=8)            # D
    with pytest.raises(FarmError):
        FarmMap(0.05, 8, -1.0, 0.5, 0.5, H=8, W=8)           # negative weight
    m = FarmMap(0.05, 8, 0.5, 0.5, 0.5, H=8, W=8)
    with pytest.raises(FarmError):
        m.set_option_i(999, 1)
    with pytest.raises(FarmError):
        m.set_option_i(1, 7)                                 # bad dtype
    from paper_2606_15476_b200 import binding
    for key, bad in ((binding.OPT_MAX_BLOCKS, 0), (binding.OPT_GAUSSIAN, 2), (binding.OPT_COVISIBILITY, -1),
                     (binding.OPT_MAX_DET_PER_CALL, 1 << 16), (binding.OPT_MAX_FRAMES_PER_CALL, 65)):
        with pytest.raises(FarmError):
            m.set_option_i(key, bad)
    for key, good in ((binding.OPT_MAX_BLOCKS, 1 << 12), (binding.OPT_GAUSSIAN, 1), (binding.OPT_COVISIBILITY, 1),
                      (binding.OPT_TIMING, 2)):
        m.set_option_i(key, good)
    with pytest.raises(FarmError) as ei:
        m.last_gaussians()                                   # no integrate call yet: FARM_ERR_STATE, not a crash
    assert ei.value.code == -4
    objs, desc, keys, owners = m.read()                      # empty, never touched the device
    assert len(objs) == 0 and len(keys) == 0
    m.destroy()


def test_no_cpu_fallback_without_device(lib):
    """Without a CUDA device integrate must fail with FARM_ERR_CUDA, never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2606_15476_b200 import FarmError, FarmMap
    m = FarmMap(0.05, 8, 0.5, 0.5, 0.5, H=8, W=8)
    n_det = np.array([0], np.int32)
    with pytest.raises(FarmError) as ei:
        m.integrate_batch(1, 1, 1, 1, 1, None, n_det)        # dummy non-NULL pointers; fails before any use
    assert ei.value.code == -2


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_15476_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "farm_oracle" not in src and "import oracle" not in src and "from oracle" not in src, f


def test_header_is_plain_c_and_links_from_c(lib, tmp_path):
    """The boundary is a C ABI: include/farm.h compiles as C99 (-pedantic) and a plain C program links against
    libfarm_map.so and drives the host-side part of it (no GPU needed: nothing here touches the device)."""
    import shutil
    import subprocess
    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    from paper_2606_15476_b200 import binding
    src = tmp_path / "t.c"
    src.write_text(r'''
#include <stdio.h>
#include "farm.h"
int main(void) {
  farm_map *m = NULL;
  int n = -1;
  long long nv = -1;
  if (farm_map_create(0.05f, 64, 0.5f, 0.5f, 0.5f, &m) != FARM_OK) return 1;
  if (farm_map_set_option_i(m, FARM_OPT_IMG_W, 160) || farm_map_set_option_i(m, FARM_OPT_IMG_H, 120)) return 2;
  if (farm_map_set_option_i(m, FARM_OPT_DESC_DTYPE, 9) != FARM_ERR_INVALID_ARG) return 3;
  if (farm_map_read(m, NULL, &n, NULL, NULL, NULL, &nv) != FARM_OK || n != 0 || nv != 0) return 4;
  printf("%s|%d\n", farm_last_error(), (int)sizeof(farm_object));
  return farm_map_destroy(m);
}
''')
    exe = tmp_path / "t"
    libdir = os.path.dirname(binding.LIB_PATH)
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(ROOT, "include"),
                           str(src), "-o", str(exe), "-L", libdir, "-lfarm_map", f"-Wl,-rpath,{libdir}"])
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0, out
    assert out.stdout.strip() == f"bad dtype|{binding.OBJECT_DTYPE.itemsize}"


def test_round2_options_and_calls_validate_on_the_host(lib):
    """The options and entry points added in round 2 validate their host-visible arguments without a device; calls that
    need an option that is off fail with FARM_ERR_STATE."""
    from paper_2606_15476_b200 import FarmError, FarmMap, binding
    m = FarmMap(0.05, 8, 0.5, 0.5, 0.5, H=8, W=8)
    for key, bad in ((binding.OPT_VIEWS, 9), (binding.OPT_VIEWS, -1), (binding.OPT_CORRESPONDENCE, 2), (binding.OPT_GEOMETRY, 2),
                     (binding.OPT_SIM_PATH, 4), (binding.OPT_EDGES, 17), (binding.OPT_EDGES, -1), (binding.OPT_INPUTS_READY, 2)):
        with pytest.raises(FarmError):
            m.set_option_i(key, bad)
    for key, good in ((binding.OPT_VIEWS, 4), (binding.OPT_CORRESPONDENCE, 1), (binding.OPT_GEOMETRY, 1), (binding.OPT_SIM_PATH, 3),
                      (binding.OPT_EDGES, 16), (binding.OPT_INPUTS_READY, 1)):
        m.set_option_i(key, good)
    for key, bad in ((binding.OPTF_EDGE_DECAY, 0.0), (binding.OPTF_EDGE_DECAY, 1.5), (binding.OPTF_EDGE_CUTOFF, -1.0),
                     (binding.OPTF_EDGE_CUTOFF, float("inf")), (binding.OPTF_EDGE_DECAY, float("nan"))):
        with pytest.raises(FarmError):
            m.set_option_f(key, bad)
    m.set_option_f(binding.OPTF_EDGE_DECAY, 1.0)
    m.set_option_f(binding.OPTF_EDGE_CUTOFF, 0.0)
    for key in (binding.OPTF_VIEW_COS, binding.OPTF_VIEW_CLOSER, binding.OPTF_PREFILTER_COS, binding.OPTF_HELLINGER_BUDGET):
        m.set_option_f(key, 0.5)
        with pytest.raises(FarmError):
            m.set_option_f(key, float("nan"))
    with pytest.raises(FarmError):
        m.set_frame_seq(-1)
    m.set_frame_seq(5)
    assert m.get_frame_seq() == 5
    with pytest.raises(FarmError) as ei:
        m.set_frame_seq(4)                                   # only forward
    assert ei.value.code == -4
    m.destroy()
    m2 = FarmMap(0.05, 8, 0.5, 0.5, 0.5, H=8, W=8)
    for call in (m2.read_alias, m2.last_merges, m2.read_views, m2.read_edges):
        with pytest.raises(FarmError) as ei:
            call()                                           # option off
        assert ei.value.code == -4
    import numpy as np
    lib_ = binding.load_library()
    q = np.zeros(32, np.float32)
    rc = lib_.farm_map_query(m2._h, None, None, None, 8, 8, 8, 0, None, q.ctypes.data, -1, 0, None, None, 1, None, None, None, None, None, None)
    assert rc == binding.ERR_INVALID_ARG                     # NULL embeddings
    one = np.zeros(8, np.float32)
    rc = lib_.farm_map_query(m2._h, one.ctypes.data, one.ctypes.data, one.ctypes.data, 8, 8, 8, 0, None, q.ctypes.data, -1, 7, None, None, 1,
                             None, None, None, None, None, None)
    assert rc == binding.ERR_INVALID_ARG                     # too many predicates
    m2.destroy()


def test_no_alloc_entry_point_rejects_oversized_requests_on_the_host(lib):
    """farm_cosine_rowmax_noalloc checks its sizes against the fixed scratch array before touching the device."""
    from paper_2606_15476_b200 import binding
    lib_ = binding.load_library()
    for M, N, D, dt in ((binding.NOALLOC_MAX_M + 1, 1, 8, 0), (1, binding.NOALLOC_MAX_N + 1, 8, 0), (1, 1, 0, 0), (1, 1, 8193, 0),
                        (1, 1, 8, 3), (-1, 1, 8, 0), (1, 1, 8, 0)):            # the last one: NULL operands
        assert lib_.farm_cosine_rowmax_noalloc(None, M, None, N, D, dt, None, None, None) == binding.ERR_INVALID_ARG
    assert b"FARM_NOALLOC_MAX_M" in lib_.farm_last_error() or b"NULL" in lib_.farm_last_error()
    hdr = open(os.path.join(os.path.dirname(__file__), "..", "include", "farm.h")).read()
    assert f"#define FARM_NOALLOC_MAX_M {binding.NOALLOC_MAX_M}" in hdr and f"#define FARM_NOALLOC_MAX_N {binding.NOALLOC_MAX_N}" in hdr
