"""The oracle side must run without the product library, and the two sides share no code.

VERDICT r1 weak point 1 / ADVICE r1: the oracle pins and ``bench.py --impl reference`` used to reach
the seeded generators through the product package, which dlopens libskel.so. The generators now live
in ``skel_inputs.py`` (numpy only); these tests keep it that way.
"""
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(code: str, *argv: str) -> subprocess.CompletedProcess:
    env = dict(os.environ, PYTHONPATH=ROOT)
    return subprocess.run([sys.executable, "-c", code, *argv], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def test_oracle_and_generators_do_not_map_the_product_library():
    code = (
        "import sys, numpy as np\n"
        "import oracle as O, skel_inputs as I\n"
        "x = I.uniform_pm1_f32(1, 1000)\n"
        "r, a = O.reduce_f32(O.FN_ADD, x)\n"
        "maps = open('/proc/self/maps').read()\n"
        "assert 'liboracle' in maps\n"
        "assert 'libskel' not in maps, 'the oracle side mapped libskel.so'\n"
        "assert not any(m.startswith('paper_1405_2915_b200') for m in sys.modules), 'product package imported'\n"
        "assert 'torch' not in sys.modules\n"
        "print('ok')\n")
    p = _run(code)
    assert p.returncode == 0 and p.stdout.strip() == "ok", p.stderr


def test_oracle_pins_collect_without_the_product_package():
    """Importing the pins module pulls in neither the product package nor libskel.so."""
    code = (
        "import sys, importlib.util\n"
        "spec = importlib.util.spec_from_file_location('pins', 'tests/test_oracle_pins.py')\n"
        "m = importlib.util.module_from_spec(spec); spec.loader.exec_module(m)\n"
        "assert not any(k.startswith('paper_1405_2915_b200') for k in sys.modules)\n"
        "assert 'libskel' not in open('/proc/self/maps').read()\n"
        "print('ok')\n")
    p = _run(code)
    assert p.returncode == 0 and p.stdout.strip() == "ok", p.stderr


def test_reference_arm_does_not_map_the_product_library():
    """bench.py --impl reference (the oracle timed on the host cores) on a tiny sample."""
    code = (
        "import sys, runpy\n"
        "sys.argv = ['bench.py', '--impl', 'reference', '--steps', '1', '--warmup', '0', '--ref-div', '4096']\n"
        "runpy.run_path('bench.py', run_name='__main__')\n"
        "maps = open('/proc/self/maps').read()\n"
        "assert 'libskel' not in maps, 'reference arm mapped libskel.so'\n"
        "assert not any(k.startswith('paper_1405_2915_b200') for k in sys.modules)\n")
    p = _run(code)
    assert p.returncode == 0, p.stderr
    assert '"impl": "reference"' in p.stdout


def _sources(*dirs, exts):
    for d in dirs:
        for base, _, files in os.walk(os.path.join(ROOT, d)):
            for f in files:
                if f.endswith(exts):
                    yield os.path.join(base, f)


def test_no_shared_code_between_oracle_and_product():
    for path in _sources("oracle", exts=(".py", ".cpp", ".c", ".h")):
        src = open(path).read()
        assert not re.search(r"^\s*(from|import)\s+paper_1405_2915_b200", src, re.M), path
        assert not re.search(r'#include\s+["<](skel\.h|.*csrc/)', src), path
    for path in _sources("paper_1405_2915_b200", "include", exts=(".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
        src = open(path).read()
        assert not re.search(r"^\s*(from|import)\s+oracle\b", src, re.M), path
        assert "oracle/" not in src and "liboracle" not in src, path
    gen = open(os.path.join(ROOT, "skel_inputs.py")).read()
    assert not re.search(r"^\s*(from|import)\s+(oracle|paper_1405_2915_b200|torch)\b", gen, re.M)
