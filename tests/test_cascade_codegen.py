"""Split / Cascade / Assemble / Emit of Alg 2.1 as a build-time generator (gen/cascade.py):
  * the augmented systems it DERIVES from the declared conservation laws (trackers, chain rule, lattice scaling) equal the
    oracle's independently hand-derived flux/source at random states -- for all 16 systems of the library: ADR, Allen-Cahn,
    weakly compressible NSE, NSF 2D (conserved-field trackers + chain rule), MHD 2D (+ Powell source), NSF 3D (derived-parent
    trackers), HCNSF (symmetric-gradient combination trackers + prescribed fields), MHD 3D (curl trackers), and the
    tracker-free ones (advection, Burgers, SWE flat / over a bed, Euler, URF, Maxwell, elasticity);
  * the committed csrc/cascade_generated.cuh is what the generator emits (byte for byte);
  * the emitted C++ evaluated on the HOST through the C-ABI hook lbmk_generated_flux gives the same numbers.
CPU only; the device-side self-check of the hand-written delta forms against the emitted code is in tests/test_gpu_round2.py."""
import os

import numpy as np
import pytest

import oracle
from paper_2607_05668_b200.gen import cascade as G

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CASES = {   # system -> (params, sample state maker)
    "euler2d": ([1.4], lambda r: np.array([1.2, 0.3, -0.2, 3.0]) * (1 + 0.1 * r.standard_normal(4))),
    "swe2d_bathy": ([9.81], lambda r: np.array([0.9, 0.2, -0.1]) * (1 + 0.1 * r.standard_normal(3))),
    "adr2d": ([0.1, -0.1, 0.01, 1.0], lambda r: np.array([0.4, 0.02, -0.03]) * (1 + 0.1 * r.standard_normal(3))),
    "allencahn2d": ([0.01, 1.0], lambda r: np.array([0.3, 0.02, -0.03]) * (1 + 0.1 * r.standard_normal(3))),
    "inse2d": ([1.7, 5e-3], lambda r: np.concatenate([[1.1, 0.2, -0.3], 0.05 * r.standard_normal(4)])),
    "nsf2d": ([1.4, 2e-3, 1e-2], lambda r: np.concatenate([[1.3, 0.4, -0.9, 3.1], 0.05 * r.standard_normal(8)])),
    "mhd2d": ([1.4, 2e-3, 1e-2, 5e-3], lambda r: np.concatenate([[1.3, 0.4, -0.9, 3.5, 0.6, -0.3], 0.05 * r.standard_normal(12)])),
    "nsf3d": ([1.4, 2e-3, 1e-2], lambda r: np.concatenate([[1.3, 0.4, -0.9, 0.5, 3.1], 0.05 * r.standard_normal(12)])),
    "advection2d": ([0.7, -0.4], lambda r: np.array([0.8]) * (1 + 0.1 * r.standard_normal(1))),
    "burgers2d": ([], lambda r: np.array([0.6]) * (1 + 0.1 * r.standard_normal(1))),
    "swe2d": ([9.81], lambda r: np.array([0.9, 0.2, -0.1]) * (1 + 0.1 * r.standard_normal(3))),
    "urf2d": ([], lambda r: np.array([3.0, 0.8, -0.5]) * (1 + 0.1 * r.standard_normal(3))),
    "maxwell2d": ([1.3], lambda r: np.array([0.3, 0.2, -0.4]) * (1 + 0.1 * r.standard_normal(3))),
    "elasticity2d": ([1.1, 0.8, 1.4], lambda r: np.array([1.05, 0.03, -0.02, 0.97, 0.1, -0.2]) * (1 + 0.05 * r.standard_normal(6))),
    # reduced symmetric-gradient basis with the prescribed alpha / u_s fields
    "hcnsf3d": ([1.4, 2e-3, 1e-2, 0.1], lambda r: np.concatenate([[1.3, 0.4, -0.9, 0.5, 3.1], 0.05 * r.standard_normal(9)])),
    # current-density trackers J = curl B (C5)
    "mhd3d": ([1.4, 5e-3], lambda r: np.concatenate([[1.3, 0.4, -0.9, 0.5, 3.6, 0.6, -0.3, 0.2], 0.05 * r.standard_normal(3)])),
}
AUX = np.array([0.3, -0.2, 0.1, 0.05])     # alpha / u_s of HCNSF, bed slopes of SWE (first two)
MAKERS = {mk.__name__: mk for mk in G.SYSTEMS}
DX, LAM, GTAU = 0.02, 5.0, 4.0


@pytest.mark.parametrize("system", sorted(CASES))
def test_derived_augmented_system_equals_the_oracles_hand_derivation(system):
    params, mk_state = CASES[system]
    laws, fn = G.numeric(MAKERS[system])
    dim = laws.dim
    o = oracle.OracleGrid(system, 4, 4, 4 if dim == 3 else 1, DX, LAM, params=params, g_tau=GTAU)
    r = np.random.default_rng(3)
    for _ in range(5):
        U = mk_state(r)
        A = AUX
        Fo, So = o.flux_source(U, A)
        Fg, Sg = fn(U, A, params, DX, DX / LAM, GTAU)
        scale = max(np.abs(Fo).max(), np.abs(So).max())
        assert np.abs(Fg - Fo[:, :dim]).max() <= 1e-13 * scale and np.abs(Sg - So).max() <= 1e-13 * scale
    o.close()


def test_cascade_registers_the_trackers_the_paper_lists():
    """Tracker sets of SM4 (state-component lists L799-L1019): ADR (c; G_c), NSE (rho, m; G_m 2x2), NSF 2D (4 + 8: gradients of
    rho, rho u, E, L961), MHD 2D (6 + 12, L1003-L1005); with `track`: NSF 3D's derived parents u (9) and T (3)."""
    sizes = {mk.__name__: G.cascade(mk()).m for mk in G.SYSTEMS}
    assert sizes == {"euler2d": 4, "swe2d_bathy": 3, "adr2d": 3, "allencahn2d": 3, "inse2d": 7, "nsf2d": 12, "mhd2d": 18, "nsf3d": 17,
                     "advection2d": 1, "burgers2d": 1, "swe2d": 3, "urf2d": 3, "maxwell2d": 3, "elasticity2d": 6, "hcnsf3d": 14, "mhd3d": 11}
    assert len(sizes) == 16 and set(sizes) == set(oracle.SYSTEM_ID)        # every system of the library has a generated form
    aug = G.cascade(G.nsf2d())
    assert sorted(aug.names[4:]) == sorted(f"G_{v}_{b}" for v in ("rho", "m0", "m1", "E") for b in range(2))


def test_generated_header_is_what_the_generator_emits():
    with open(os.path.join(ROOT, "paper_2607_05668_b200", "csrc", "cascade_generated.cuh")) as fh:
        assert fh.read() == G.generate_text()


@pytest.mark.parametrize("system", sorted(CASES))
def test_emitted_code_on_the_host_through_the_c_abi(system):
    """lbmk_generated_flux runs the EMITTED C++ (compiled into liblbmk.so) on the host: equal to the SymPy evaluation of the same
    derivation and to the oracle."""
    import paper_2607_05668_b200 as P
    params, mk_state = CASES[system]
    laws, fn = G.numeric(MAKERS[system])
    o = oracle.OracleGrid(system, 4, 4, 4 if laws.dim == 3 else 1, DX, LAM, params=params, g_tau=GTAU)
    r = np.random.default_rng(4)
    U = mk_state(r)
    A = AUX
    F, S = P.lbmk_generated_flux(P.SYSTEM_ID[system], U, A, params, DX, LAM, GTAU, len(U))
    Fo, So = o.flux_source(U, A)
    Fg, Sg = fn(U, A, params, DX, DX / LAM, GTAU)
    scale = max(np.abs(Fo).max(), np.abs(So).max())
    assert np.abs(F - Fo).max() <= 1e-13 * scale and np.abs(S - So).max() <= 1e-13 * scale
    assert np.abs(F[:, :laws.dim] - Fg).max() <= 1e-13 * scale and np.abs(S - Sg).max() <= 1e-13 * scale
    o.close()


def test_generated_flux_misuse_is_refused():
    import paper_2607_05668_b200 as P
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_generated_flux(P.SYSTEM_ID["urf2d"], [3.0, 1.0, 1.0], None, [1.0], DX, LAM, GTAU, 3)      # URF takes no parameters
    assert e.value.status == 1
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_generated_flux(P.SYSTEM_ID["euler2d"], [1.0, 0.0, 0.0, 2.5], None, [1.4], DX, -1.0, GTAU, 4)
    assert e.value.status == 1
