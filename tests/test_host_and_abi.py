"""CPU-only checks of the boundary and the host logic: the C-ABI library builds/loads and exports every
symbol include/hz.h declares, the ctypes structs match the header, compute calls fail loudly without a
GPU (no CPU fallback), and the N>1 aggregation of bench.py works over gloo with world_size 2."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2606_21695_b200 import build
    return build.build()


def test_library_exports_every_declared_symbol(libpath):
    hdr = open(os.path.join(ROOT, "include", "hz.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(hz_[a-z_0-9]+)\s*\(", hdr))
    assert {"hz_mesh_setup", "hz_partition", "hz_ddm_solve", "hz_residual"} <= declared
    lib = ctypes.CDLL(libpath)
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in hz.h but not exported"
    from paper_2606_21695_b200 import hz
    assert set(hz.EXPORTS) == declared


def test_library_exports_every_symbol_of_the_3d_header(libpath, tmp_path):
    hdr = open(os.path.join(ROOT, "include", "hz3.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(hz3_[a-z_0-9]+)\s*\(", hdr))
    lib = ctypes.CDLL(libpath)
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in hz3.h but not exported"
    from paper_2606_21695_b200 import hz3
    assert set(hz3.EXPORTS) == declared
    src = tmp_path / "sz3.c"
    src.write_text('#include <stdio.h>\n#include "hz3.h"\nint main(void){printf("%zu %zu %zu\\n", sizeof(hz3_part_info),'
                   ' sizeof(hz3_solve_opts), sizeof(hz3_solve_info));return 0;}\n')
    exe = tmp_path / "sz3"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    a, b, c = map(int, subprocess.check_output([str(exe)]).split())
    assert (a, b, c) == (ctypes.sizeof(hz3.hz3_part_info), ctypes.sizeof(hz3.hz3_solve_opts),
                         ctypes.sizeof(hz3.hz3_solve_info))


def test_ctypes_structs_match_header_sizes(libpath, tmp_path):
    """Compile a tiny C program against include/hz.h and compare sizeof() with the ctypes mirrors."""
    from paper_2606_21695_b200 import hz
    src = tmp_path / "sz.c"
    names = ["hz_part_info", "hz_part_flags", "hz_solve_opts", "hz_solve_info", "hz_sources_info", "hz_gmres_opts",
             "hz_gmres_info", "hz_mixed_opts", "hz_mixed_info", "hz_minres_opts", "hz_minres_info"]
    body = "".join(f'printf("%zu\\n", sizeof({n}));' for n in names)
    src.write_text('#include <stdio.h>\n#include "hz.h"\nint main(void){' + body + 'return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    sizes = list(map(int, subprocess.check_output([str(exe)]).split()))
    assert sizes == [ctypes.sizeof(getattr(hz, n)) for n in names]


def test_argument_errors_need_no_gpu(libpath):
    from paper_2606_21695_b200 import hz
    c = np.ones((5, 5))
    for kwargs, status in ((dict(p=9), hz.HZ_EUNSUPPORTED), (dict(nx=0), hz.HZ_EINVAL), (dict(omega=-1.0), hz.HZ_EINVAL)):
        a = dict(nx=2, ny=2, x0=0.0, y0=0.0, x1=1.0, y1=1.0, p=2, c_nodes=c, omega=3.0, f_re=c)
        a.update(kwargs)
        with pytest.raises(hz.HzError) as e:
            hz.hz_mesh_setup(**a)
        assert e.value.status == status
    with pytest.raises(hz.HzError) as e:   # non-positive wave speed
        hz.hz_mesh_setup(2, 2, 0, 0, 1, 1, 2, np.zeros((5, 5)), 3.0, c)
    assert e.value.status == hz.HZ_EINVAL
    hz.hz_destroy(None)  # NULL-safe


def test_compute_fails_loudly_without_a_gpu(libpath):
    """No CPU fallback: on a box without a CUDA device the product path must raise, not compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for GPU-less boxes")
    from paper_2606_21695_b200 import hz
    c = np.ones((5, 5))
    with pytest.raises(hz.HzError) as e:
        hz.hz_mesh_setup(2, 2, 0, 0, 1, 1, 2, c, 3.0, c)
    assert e.value.status in (hz.HZ_ECUDA, hz.HZ_ENOMEM)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_21695_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "hz_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f
    txt = open(os.path.join(ROOT, "oracle", "hz_oracle.py")).read()
    assert "import paper_2606_21695_b200" not in txt and "from paper_2606_21695_b200" not in txt


def _gloo_worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r took (10 + 5 r) ms for 1e6 units: the job value divides by the SLOWEST rank's time
    val, max_ms = bench.job_value(1.0e6, 10.0 + 5.0 * rank, world, "cpu")
    q.put((rank, val, max_ms))
    dist.destroy_process_group()


def test_replica_aggregation_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, val, max_ms in res:
        assert max_ms == 15.0
        assert abs(val - 2 * 1.0e6 / 15.0e-3) < 1e-6 * val


def test_reference_arm_prints_contract_line():
    out = subprocess.check_output([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                                   "--warmup", "0", "--config", "2", "--n", "16"], cwd=ROOT, text=True, timeout=600)
    import json
    line = json.loads(out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
    assert line["cpu_baseline"]["cores"] == os.cpu_count()          # one oracle process per host core


def test_the_oracle_window_of_bench_reproduces_the_full_problem():
    """bench.py times the oracle on the lower-left window of the workload's subdomains (a full-size config-5 oracle
    state would be 65 536 subdomains); a subdomain's DDM cycle in the window is that of the full problem."""
    sys.path.insert(0, ROOT)
    import bench
    from oracle import hz_oracle as O
    from paper_2606_21695_b200.inputs import make_config
    inp = make_config(3, n=48)                                      # 6x6 subdomains of 8x8 elements
    w = bench._oracle_window(inp, 2)
    pr = O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega, inp.f_re.astype(complex))
    st = O.ddm_setup(pr, inp.sx, inp.sy, inp.cfl_frac)
    prw = O.Problem(w["nx"], w["ny"], w["p"], w["x0"], w["y0"], w["x1"], w["y1"], w["c"], w["omega"], w["f"].astype(complex))
    n_t = O.choose_nt(w["p"], w["hx"], w["hy"], w["c_max"], w["omega"], w["cfl"])
    assert n_t == st.tab.n_t
    stw = O.ddm_setup(prw, w["sx"], w["sy"], w["cfl"], n_t=n_t)
    for lw, l in ((0, 0), (1, 1), (2, inp.sx), (3, inp.sx + 1)):
        uw, _ = O.ddm_cycle(stw, lw, 2, True)
        u, _ = O.ddm_cycle(st, l, 2, True)
        assert np.linalg.norm(uw - u) <= 1e-12 * np.linalg.norm(u)
