"""The oracles once under AddressSanitizer + UndefinedBehaviorSanitizer: small problems with hanging nodes,
two species on two grids, every entry point the parity tests use; the sanitizers abort the child process on any finding."""
import os
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _asan_runtime():
    out = subprocess.run(["g++", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    return out if os.path.isabs(out) and os.path.exists(out) else None


@pytest.mark.parametrize("src,driver", [
    ("landau_oracle.cpp", """
        from oracle import oracle as O
        from paper_2209_03228_b200 import workloads as W
        O._LIB = LIB
        cfg = W.tiny_config("quadtree", 2, batch=1)
        o = O.Oracle(cfg["grids"], cfg["species"], 2)
        f = W.make_batch_f(cfg, [o.dof_coords(g) for g in range(o.G)], batch=1)[0]
        o.jacobian(f, 0.5); o.apply(f); o.inner(f); o.mass(0); o.pattern(1); o.ip_table(0)
        for mesh, k in ((W.semicircle_mesh(2.0, 1, 1), 3), (W.semicircle_triangles(2.0, 1, 1), 4)):
            u = O.Oracle.from_meshes([mesh], [dict(mass=1.0, charge=-1.0, grid=0)], k)
            fu = W.make_batch_f(dict(index=87, species=[dict(mass=1.0, charge=-1.0, grid=0)], state="shifted", alpha=[1.0], batch=1),
                                [u.dof_coords(0)], batch=1)[0]
            u.jacobian(fu, 0.5); u.apply(fu)
        print("sanitized run ok")
     """),
    ("landau3v_oracle.cpp", """
        from oracle import oracle3v as O
        from paper_2209_03228_b200 import workloads as W
        O._LIB = LIB
        cfg = W.config3v("tiny", batch=1)
        o = O.Oracle3V(cfg["grids"], cfg["species"])
        f = W.make_batch_f3v(cfg, [o.dof_coords(g) for g in range(o.G)], batch=1)[0]
        o.jacobian(f, 0.5); o.apply(f); o.inner(f); o.mass(0); o.fields(f, 1); o.pattern(0)
        print("sanitized run ok")
     """)])
def test_oracle_under_asan_ubsan(tmp_path, src, driver):
    rt = _asan_runtime()
    if rt is None:
        pytest.skip("no libasan runtime next to g++")
    lib = str(tmp_path / (src.replace(".cpp", "") + "_san.so"))
    subprocess.check_call(["g++", "-std=c++17", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
                           "-fno-sanitize-recover=undefined", "-shared", "-fPIC", "-o", lib, os.path.join(ROOT, "oracle", src)])
    code = "import sys\nsys.path.insert(0, %r)\nLIB = %r\n" % (ROOT, lib) + textwrap.dedent(driver)
    code = code.replace("O._LIB = LIB", "O._LIB = LIB\nO.build = lambda force=False: LIB")
    env = dict(os.environ, LD_PRELOAD=rt, ASAN_OPTIONS="detect_leaks=0", OMP_NUM_THREADS="2")
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0 and "sanitized run ok" in out.stdout, (out.stdout[-1500:], out.stderr[-3000:])
