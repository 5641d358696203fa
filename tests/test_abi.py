"""CPU-side checks of the boundary: the C-ABI library builds (nvcc cross-compiles), loads and exports every symbol
include/dem.h declares; the host logic of dem_create / dem_create_shape; and that nothing computes without a GPU.
No kernel is launched here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import dem_inputs as di

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    import paper_1607_02427_b200 as p

    p.build.build()
    p.lib()
    return p


def _declared(header_name):
    header = open(os.path.join(ROOT, "include", header_name)).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    return set(re.findall(r"\b(dem_[a-z0-9_]+)\s*\(", header))


def test_library_exports_every_declared_symbol(pkg):
    """include/dem.h is the paper's problem statement; include/dem_bench.h holds the measurement hooks."""
    declared, bench = _declared("dem.h"), _declared("dem_bench.h")
    assert declared == set(pkg.EXPORTS), declared ^ set(pkg.EXPORTS)
    assert bench == set(pkg.EXPORTS_BENCH), bench ^ set(pkg.EXPORTS_BENCH)
    assert not any(w in n for n in declared for w in ("timing", "flush", "peak", "launch_count", "swept"))
    lib = pkg.lib()
    for name in declared | bench:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.dem_version()


def test_library_is_built_from_the_sources_in_the_tree(pkg):
    """A prebuilt .so that lags any file under csrc/ or include/ must not be used silently: the hash of the sources is
    compiled into the library and build.stale() / binding.lib() compare it with the tree."""
    assert not pkg.build.stale()
    assert pkg.build.source_hash().encode() in pkg.lib().dem_version()
    names = {os.path.basename(f) for f in pkg.build.sources() + pkg.build.headers()}
    assert {"dem_fast.cuh", "dem_kernels.cuh", "dem_math.cuh", "dem_lib.cu", "dem.h", "dem_bench.h"} <= names


def test_no_torch_types_in_the_abi():
    header = open(os.path.join(ROOT, "include", "dem.h")).read()
    assert "torch" not in re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    assert 'extern "C"' in header


def test_binary_is_sm_100a(pkg):
    import shutil
    import subprocess

    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", pkg.build.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_create_and_argument_validation(pkg):
    lib = pkg.lib()
    ctx = C.c_void_p()
    assert lib.dem_create(C.byref(ctx), 4, C.c_double(1.0), 0, None) == pkg.binding.DEM_EINVAL
    assert lib.dem_create(C.byref(ctx), 3, C.c_double(-1.0), 0, None) == pkg.binding.DEM_EINVAL
    assert lib.dem_create(C.byref(ctx), 3, C.c_double(1.0), 7, None) == pkg.binding.DEM_EINVAL
    assert lib.dem_create(None, 3, C.c_double(1.0), 0, None) == pkg.binding.DEM_EINVAL
    assert lib.dem_create(C.byref(ctx), 3, C.c_double(1.0), 0, None) == 0 and ctx.value
    assert lib.dem_set_eps_par(ctx, C.c_double(-1.0)) == pkg.binding.DEM_EINVAL
    assert lib.dem_get_neighbors(ctx, None, None, None, None) == pkg.binding.DEM_ESTALE
    assert b"no neighbour list" in lib.dem_last_error(ctx)
    assert lib.dem_destroy(ctx) == 0


def test_shape_validation_host_logic(pkg):
    d = pkg.Dem(3, 1.0, "f32", stream=0)
    for s in (di.cube(), di.octahedron(), di.tetrahedron(), di.truncated_icosahedron(), di.icosahedron(),
              di.sphere(0.2), di.rod(1.0, 0.1), di.triangular_plate()):
        d.create_shape_dict(s)
    assert d.shapes == list(range(8))
    with pytest.raises(pkg.DemError):  # DEM_MAX_SHAPES
        d.create_shape_dict(di.cube())
    d.close()
    d = pkg.Dem(3, 1.0, "f64", stream=0)
    cube = di.cube()
    bad = [
        dict(verts=cube["verts"], faces=[[0, 1, 99]], rounding=0.1),                      # index out of range
        dict(verts=cube["verts"], faces=[[0, 1]], rounding=0.1),                          # < 3 vertices
        dict(verts=cube["verts"], faces=[[0, 1, 3, 6]], rounding=0.1),                    # not planar
        dict(verts=[[0, 0, 0], [2, 0, 0], [0.5, 0.2, 0], [1, 2, 0], [-1, 1, 0]], faces=[[0, 1, 2, 3, 4]], rounding=0.1),
        dict(verts=cube["verts"], faces=cube["faces"], rounding=0.0),                     # rounding <= 0
        dict(verts=cube["verts"], faces=cube["faces"], rounding=0.1, mass=0.0),
        dict(verts=cube["verts"], faces=cube["faces"], edges=[[0, 8]], rounding=0.1),
        dict(verts=np.zeros((0, 3)), rounding=0.1),
    ]
    for kw in bad:
        with pytest.raises(pkg.DemError) as e:
            d.create_shape(**kw)
        assert e.value.code == pkg.binding.DEM_EINVAL, kw
    # either face orientation is accepted (faces are two-sided), edges are derived from the faces
    d.create_shape(cube["verts"], [list(reversed(f)) for f in cube["faces"]], None, 0.1)
    d.close()
    d2 = pkg.Dem(2, 1.0, "f32", stream=0)
    with pytest.raises(pkg.DemError):
        d2.create_shape(cube["verts"], cube["faces"], None, 0.1)  # faces in 2D
    d2.create_shape_dict(di.square())
    d2.create_shape_dict(di.disk(0.1))
    d2.close()


def test_no_cpu_path(pkg):
    """Without a device the computing calls fail loudly (DEM_ECUDA / TypeError), they do not fall back."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less box")
    d = pkg.Dem(3, 1.0, "f32", stream=0)
    d.create_shape_dict(di.cube())
    st = di.make_config(2, scale=4)
    pos = torch.tensor(st["pos"], dtype=torch.float32)
    sid = torch.tensor(st["shape_id"], dtype=torch.int32)
    with pytest.raises(TypeError):
        d.build_neighbors(pos, sid, st["box"], st["r_cut"])
    n = st["N"]
    host = [np.zeros((n, 4), dtype=np.float32) for _ in range(4)]
    with pytest.raises(pkg.DemError) as e:
        d.compute_host(host[0], host[1], np.zeros(n, dtype=np.int32), st["box"], st["r_cut"], host[2], host[3])
    assert e.value.code in (pkg.binding.DEM_ECUDA, pkg.binding.DEM_ENOMEM)
    d.close()


def test_product_does_not_import_the_oracle():
    """The product path shares nothing with the oracle: no file under the package or bench's GPU arm imports it."""
    pk = os.path.join(ROOT, "paper_1607_02427_b200")
    for dirpath, _, files in os.walk(pk):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "dem_oracle" not in src and "oracle/" not in src and "from oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1607_02427_b200" not in src and "libdem_b200" not in src and "csrc" not in src
