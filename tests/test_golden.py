"""The paper's printed values (tests/golden/paper_constants.txt, each with its citation) against the
oracle's defaults, the binding's defaults and the arithmetic DESIGN.md derives from them."""
from pathlib import Path

import math

import numpy as np

GOLD = Path(__file__).resolve().parent / "golden" / "paper_constants.txt"


def _gold():
    out = {}
    for line in GOLD.read_text().splitlines():
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split()
            out[k] = float(v)
    return out


def test_defaults_are_the_papers(oracle):
    g = _gold()
    from paper_2510_13726_b200 import binding as B, inputs as I
    for make in (oracle.make_params, B.make_params):
        p = make(4, 4, 4)
        assert p.kappa == g["kappa"] and p.E == g["E"]
        assert p.newton_tol == g["newton_tol"] and p.newton_max_iter == int(g["newton_max_iter"])
    assert I.DEFAULTS["kappa"] == g["kappa"] and I.DEFAULTS["E"] == g["E"]


def test_truncated_spalding_is_eq17(oracle):
    """Eq. 17/18 retyped from the paper's constants: f(u_tau) = u+ + (e^{k u+} - sum of the
    first four Taylor terms)/E - y u_tau/nu, at values where each term matters."""
    g = _gold()
    k, E = g["kappa"], g["E"]
    for U, ut, y, nu in [(0.05, 0.0025, 2.75, 3.2e-4), (0.04, 0.004, 3.0, 6.0e-5), (1e-3, 5e-4, 2.1, 1e-3)]:
        up = U / ut
        taylor = sum((k * up) ** m / math.factorial(m) for m in range(int(g["spalding_terms"])))
        expect = up + (np.exp(k * up) - taylor) / E - y * ut / nu
        assert abs(oracle.spalding_f(ut, U, y, nu) - expect) <= 1e-12 * max(1.0, abs(expect))


def test_table1_byte_accounting():
    """Table 1: 152 B = read + write of 19 fp32 populations; 204 B adds 13 fp32 fields.
    The D3Q27 analogue used as algorithmic bytes in bench.py is 2 x 27 x 4 = 216 B."""
    g = _gold()
    assert g["rrlbm_bytes"] == 2 * 19 * 4
    assert g["hhrrlbm_bytes"] - g["rrlbm_bytes"] == 13 * 4
    import bench
    assert bench.BYTES_PER_CELL == 2 * 27 * 4
    # the paper's implied DRAM rate, quoted in BASELINE.md as context
    assert abs(g["hhrrlbm_mlups"] * g["hhrrlbm_bytes"] / 1e3 - 867.4) < 0.1
