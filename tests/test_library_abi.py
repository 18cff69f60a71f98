"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/dp.h declares, and the
host-only entry points work.  No compute call is made (there is no GPU in the CPU test container)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def dp():
    import paper_2210_01837_b200 as dp
    from paper_2210_01837_b200 import build
    build.build()
    return dp


def test_every_declared_symbol_is_exported(dp):
    hdr = open(os.path.join(ROOT, "include", "dp.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(dp_[a-z_0-9]+)\s*\(", hdr)))
    assert "dp_create" in declared and "dp_mobility_apply" in declared and "dp_destroy" in declared
    assert sorted(dp.binding.EXPORTS) == declared
    assert sorted(dp.exported_symbols()) == declared


def test_host_only_entry_points(dp):
    L = dp.load_library()
    assert L.dp_strerror(0) == b"ok" and L.dp_strerror(-5) == b"particle outside the domain"
    assert set(dp.supported_nz()) >= {16, 32, 48}
    assert L.dp_destroy(None) == 0
    assert L.dp_device_bytes(None) == 0
    # the ES normalisation is computed independently on both sides and must agree to 1e-15
    import oracle
    for alpha, beta in ((2.0, 6 * 1.714), (1.99, 6 * 1.327), (1.99, 6 * 2.216), (1.5, 4 * 1.785)):
        assert dp.es_norm(alpha, beta) == pytest.approx(oracle.es_norm(alpha, beta), rel=1e-15)


def test_effective_radius_matches_the_papers_tables(dp):
    """dp_es_radius_over_h = dp_effective_radius / h (host-side quadrature, no device, no plan) against the values the paper prints (tests/golden/paper_tables.txt:
    Tables I-II) to <= 1 %, and against eq 8's Gaussian relation through a near-Gaussian ES kernel."""
    L = dp.load_library()
    rows = []
    with open(os.path.join(ROOT, "tests", "golden", "paper_tables.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                kind, w, bw, rh = line.split()
                rows.append((kind, int(w), float(bw), float(rh)))
    assert len(rows) >= 3
    for kind, w, bw, rh in rows:
        got = L.dp_es_radius_over_h(w, bw * w, 1 if kind == "D" else 0)       # R_h / h
        assert got == pytest.approx(rh, rel=0.01), (kind, w, bw, got)
    # Table I, m = 6: monopole and dipole radii agree "to 3 digits" by construction of the table
    rm, rd = L.dp_es_radius_over_h(6, 6 * 1.327, 0), L.dp_es_radius_over_h(6, 6 * 2.216, 1)
    assert rm == pytest.approx(rd, rel=2e-3) and rm == pytest.approx(1.73, rel=0.01)
    assert L.dp_effective_radius(None, 0) < 0


def test_product_path_has_no_cpu_fallback(dp):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import workloads
    prob, pos, F, T = workloads.config(1)
    with pytest.raises(dp.DPError):
        dp.Plan(prob, max_particles=8)        # dp_create fails loudly without a device


def test_package_does_not_import_the_oracle():
    import subprocess, sys
    code = "import sys; import paper_2210_01837_b200 as dp; dp.load_library(); assert 'oracle' not in sys.modules"
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)
    src = "".join(open(os.path.join(ROOT, "paper_2210_01837_b200", f)).read() for f in ("__init__.py", "binding.py", "build.py"))
    assert "import oracle" not in src and "from oracle" not in src
