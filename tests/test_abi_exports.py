"""CPU-only checks of the boundary: the C-ABI library builds, loads, and exports every symbol include/spinllg.h declares.
No compute call is made here (there is no GPU in the build container)."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "spinllg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = re.findall(r"\b([a-z_0-9]+)\s*\(", text)
    return sorted({n for n in names if n not in ("defined",)})


def test_library_builds_and_exports_every_declared_symbol():
    import paper_1901_11350_b200 as P
    L = P.lib()
    decl = declared_functions()
    assert len(decl) >= 25
    for name in decl:
        assert hasattr(L, name), f"{name} declared in include/spinllg.h but not exported"
    assert sorted(P.EXPORTS) == decl
    assert "sm_100a" in P.version()


def test_library_is_built_for_sm_100a():
    import subprocess
    import paper_1901_11350_b200.build as B
    out = subprocess.run(["cuobjdump", "-lelf", B.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_cpu_fallback_without_device():
    """Without a CUDA device the product must fail loudly, not compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_1901_11350_b200 as P
    with pytest.raises(P.SpinError) as e:
        P.SpinSystem(np.eye(3), [[0, 0, 0]], (4, 4, 1), (1, 1, 0))
    assert e.value.code == -4 and "no CPU fallback" in str(e.value)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1901_11350_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "spin_oracle" not in src and "liboracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "spin_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_1901_11350_b200" not in osrc.replace("paper_1901_11350_b200/; only", "").replace("(paper_1901_11350_b200) never", "")


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_planner_generates_and_compiles_specialised_sweeps(cfg, monkeypatch):
    """Host planner + NVRTC (no device needed): the gather tables of every config become a translation unit that compiles
    for sm_100a.  Entry counts per spin as SURVEY 8(a) states them: 4 / 18 / 6 / 9 pairs + 4 quadruplet roles / 6."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("planner-only mode is for boxes without a GPU")
    monkeypatch.setenv("SPINLLG_PLANNER_ONLY", "1")
    import paper_1901_11350_b200 as P
    import workloads as W
    w = W.CONFIGS[cfg]()
    s = P.SpinSystem.from_workload(w, set_spins=False)
    src, nbytes = s.spin_jit_source(compile=True)
    assert nbytes > 10000
    begin = [int(x) for x in re.search(r"PAIR_BEGIN\[\d+\] = \{([^}]*)\}", src).group(1).split(",")]
    qbegin = [int(x) for x in re.search(r"QUAD_BEGIN\[\d+\] = \{([^}]*)\}", src).group(1).split(",")]
    expect_pairs = {1: [4], 2: [18], 3: [6], 4: [9, 9], 5: [6]}[cfg]
    assert [b - a for a, b in zip(begin, begin[1:])] == expect_pairs
    assert [b - a for a, b in zip(qbegin, qbegin[1:])] == ({4: [4, 4]}.get(cfg, [0] * w.n_basis))
    # computing without a device still fails loudly
    with pytest.raises(P.SpinError) as e:
        s.llg_iterate(1)
    assert e.value.code == -4


def test_header_is_plain_c_and_links_from_c(tmp_path):
    """The boundary is a C ABI: include/spinllg.h compiles as C11 with gcc, and a C program that takes the address of every declared
    function links against libspinllg.so and runs (planner-only mode: no device needed, computing calls fail with SPIN_ERR_CUDA)."""
    import shutil
    import paper_1901_11350_b200 as P
    P.lib()
    names = declared_functions()
    src = tmp_path / "use_abi.c"
    body = "    void *volatile fns[] = {" + ", ".join(f"(void *){n}" for n in names) + "};\n    for (unsigned k = 0; k < sizeof fns / sizeof fns[0]; ++k) if (!fns[k]) return 100;"
    src.write_text(f'''#include <stdio.h>
#include <string.h>
#include "spinllg.h"
int main(void) {{
{body}
    const double brav[9] = {{1, 0, 0, 0, 1, 0, 0, 0, 1}}, basis[3] = {{0, 0, 0}};
    const int cells[3] = {{4, 4, 1}}, per[3] = {{1, 1, 0}};
    spin_system *s = NULL;
    int rc = spin_geometry_create(brav, 1, basis, cells, per, 1.0, &s);
    if (rc != SPIN_OK) {{ printf("create: %d %s\\n", rc, spin_last_error()); return rc == SPIN_ERR_CUDA ? 0 : 1; }}
    if (spin_system_nspins(s) != 16) return 2;
    const int bi[1] = {{0}}, t[3] = {{1, 0, 0}};
    const double J[1] = {{1.0}};
    if (hamiltonian_set_pairs(s, 1, bi, bi, t, J, NULL) != SPIN_OK) return 3;
    if (hamiltonian_set_pairs(s, 1, bi, bi, (const int[3]){{0, 0, 0}}, J, NULL) != SPIN_ERR_ARG) return 4;      /* self pair */
    rc = llg_iterate(s, 1);                       /* no device in this test: must fail loudly, never fall back */
    printf("llg_iterate without a device: %d (%s)\\n", rc, spin_last_error());
    spin_system_destroy(s);
    return rc == SPIN_ERR_CUDA ? 0 : (rc == SPIN_OK ? 0 : 5);
}}
''')
    exe = tmp_path / "use_abi"
    libdir = os.path.dirname(P.binding.LIB_PATH) if hasattr(P, "binding") and hasattr(P.binding, "LIB_PATH") else os.path.join(ROOT, "paper_1901_11350_b200")
    cmd = ["gcc", "-std=c11", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe),
           "-L", libdir, "-lspinllg", f"-Wl,-rpath,{libdir}"]
    subprocess.run(cmd, check=True)
    env = dict(os.environ, SPINLLG_PLANNER_ONLY="1")
    r = subprocess.run([str(exe)], env=env, capture_output=True, text=True)
    assert r.returncode == 0, (r.returncode, r.stdout, r.stderr)


def test_jit_compiler_is_bound_by_path_even_with_torch_loaded():
    # torch preloads its own libnvrtc.so.12 (another version, same soname); the library must still find the toolkit's by path
    import torch  # noqa: F401
    import paper_1901_11350_b200 as P
    info = P.spin_jit_compiler_info()
    assert info.split(".")[0].isdigit(), info
    toolkit = "/usr/local/cuda/lib64/libnvrtc.so.12"
    if os.path.exists(toolkit) and not os.environ.get("SPINLLG_NVRTC"):
        assert toolkit in info, info
