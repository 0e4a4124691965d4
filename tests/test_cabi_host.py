"""CPU-side checks of the boundary: liblbmk.so builds, loads and exports every symbol include/lbmk.h declares;
host-side validation, grid scaling and the a-priori sub-characteristic check behave as documented.
No compute call is made here (there is no GPU on this box and no CPU fallback in the product)."""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest

import paper_2607_05668_b200 as P
import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "lbmk.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lbmk_[a-z_0-9A-Z]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = P.lib()
    names = declared_symbols()
    assert len(names) >= 25
    for n in names:
        assert hasattr(L, n), f"liblbmk.so does not export {n}"
    # and the binding marshals every one of them
    assert set(names) == set(P.SYMBOLS), set(names) ^ set(P.SYMBOLS)
    for n in names:
        assert callable(getattr(P, n)), f"binding lacks a wrapper named {n}"


def test_version_and_lattice_constants():
    assert "sm_100a" in P.lbmk_version()
    for lat, D in ((P.LBMK_D2Q5, 2), (P.LBMK_D3Q7, 3)):
        c, w, cs2 = P.lbmk_lattice_constants(lat)
        # Table SM1; isotropy eq (2.5)
        assert abs(w.sum() - 1) < 1e-15 and np.abs((w[:, None] * c).sum(0)).max() < 1e-15
        M2 = np.einsum("i,ia,ib->ab", w, c, c)
        assert np.allclose(M2[:D, :D], cs2 * np.eye(D), atol=1e-15)
        assert cs2 == {2: 1 / 3, 3: 1 / 4}[D]


def test_system_info_matches_workloads():
    for name, sid in P.SYSTEM_ID.items():
        s = P.System(name, params=_params(name), tau_R=1.0, g_tau=3.0)
        assert s.m_total == len(W.COMPONENTS[name]) and s.m_conserved == W.N_CONSERVED[name]
        assert s.Q == (5 if W.LATTICE_OF[name] == "D2Q5" else 7)
        assert s.n_aux == len(W.AUX_FIELDS.get(name, []))          # prescribed coefficient fields
        s.close()


def _params(name):
    return {"advection2d": [0.1, 0.05], "burgers2d": [], "swe2d": [1.0], "euler2d": [1.4], "adr2d": [0.1, -0.1, 0.01, 1.0],
            "nsf3d": [1.4, 1e-3, 5e-3], "mhd3d": [1.4, 1e-3], "urf2d": [], "maxwell2d": [1.0], "allencahn2d": [0.01, 1.0], "inse2d": [1.0, 0.01], "elasticity2d": [1.0, 1.0, 2.0], "nsf2d": [1.4, 0.0084, 0.0416],
            "swe2d_bathy": [10.0], "hcnsf3d": [1.4, 1e-2, 1e-2, 1e-3], "mhd2d": [1.4, 0.01, 0.01, 0.01]}[name]


def test_argument_validation():
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_system_create(99, P.LBMK_D2Q5, [])
    assert e.value.status == 1
    with pytest.raises(P.LbmkError):
        P.lbmk_system_create(P.SYSTEM_ID["euler2d"], P.LBMK_D3Q7, [1.4])      # lattice / dimension mismatch
    with pytest.raises(P.LbmkError):
        P.lbmk_system_create(P.SYSTEM_ID["euler2d"], P.LBMK_D2Q5, [1.4, 2.0])  # wrong parameter count
    s = P.System("nsf3d", params=_params("nsf3d"), tau_R=20.0, g_tau=3.0)
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_system_set_reference(s.h, [1, 0.1, 0, 0, 2] + [0] * 12)         # moving reference unsupported
    assert e.value.status == 6
    with pytest.raises(P.LbmkError):
        P.lbmk_system_set_omega(s.h, [2.5])
    with pytest.raises(P.LbmkError):
        P.lbmk_system_set_mms(s.h, 1, [0.1])                                    # wrong mms parameter count
    with pytest.raises(P.LbmkError):
        P.lbmk_grid_create(s.h, 8, 8, 0, 0, 0.1, 5.0, P.LBMK_F64, 0)
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_grid_create(s.h, 2048, 1024, 1024, 0, 0.1, 5.0, P.LBMK_F32_SHIFTED, 0)   # 2^31 nodes: above the maximum
    assert e.value.status == 1
    g = P.lbmk_grid_create(s.h, 2047, 1024, 1024, 0, 0.1, 5.0, P.LBMK_F32_SHIFTED, 0)    # largest accepted size class
    assert P.lbmk_grid_workspace_bytes(g) > 2 * 17 * 7 * 2047 * 1024 * 1024 * 4          # > 2 TB: size_t arithmetic, no overflow
    P.lbmk_grid_destroy(g)
    e2 = P.System("euler2d", params=[1.4], tau_R=1.0)
    with pytest.raises(P.LbmkError):
        P.lbmk_grid_create(e2.h, 8, 8, 2, 0, 0.1, 5.0, P.LBMK_F64, 0)           # nz != 1 in 2D
    with pytest.raises(P.LbmkError):
        P.lbmk_grid_create(e2.h, 8, 8, 1, P.LBMK_DIRICHLET_MMS, 0.1, 5.0, P.LBMK_F64, 0)   # bounded needs MMS


def test_grid_scaling_and_workspace_layout():
    """omega_k = 1/(1/2 + tau_R dt) for conserved fields (L194), 1/(g_tau + 1) for trackers (L718); workspace
    = populations (x2 for the two-lattice pattern) + small tables + the per-row forcing coefficients."""
    w = W.c4_nsf3d(16)
    s = P.System(w.system, params=w.params, tau_R=w.tau_R, g_tau=w.g_tau, U_ref=w.U_ref, mms_id=1, mms_params=w.mms_params)
    g = P.lbmk_grid_create(s.h, 16, 16, 16, 0, w.dx, w.lam, P.LBMK_F32_SHIFTED, 0)
    om = P.lbmk_grid_omega(g, 17)
    assert np.allclose(om[:5], 1.0 / (0.5 + w.tau_R * w.dt), rtol=1e-15) and np.allclose(om[5:], 1.0 / (w.g_tau + 1.0))
    pops = 17 * 7 * 16 ** 3 * 4
    P.lbmk_grid_set_option(g, P.LBMK_OPT_PATTERN, P.LBMK_PATTERN_PULL2)
    b2 = P.lbmk_grid_workspace_bytes(g)
    P.lbmk_grid_set_option(g, P.LBMK_OPT_PATTERN, P.LBMK_PATTERN_AA)
    b1 = P.lbmk_grid_workspace_bytes(g)
    small = 65536 + 2 * 64 * 16 * 16 * 128 * 4   # tables, scratch, forcing coefficients: 2 buffers x <= 64 steps x [ny*nz][NC <= 128]
    assert 2 * pops <= b2 < 2 * pops + small and pops <= b1 < pops + small
    assert b2 - b1 == pops                     # the second lattice is the only difference
    assert P.lbmk_time(g) == (0, 0.0)
    # calls out of order are refused, not crashed
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_step(g, 1)
    assert e.value.status == 5
    with pytest.raises(P.LbmkError):
        P.lbmk_grid_bind_workspace(g, 0, b1)
    with pytest.raises(P.LbmkError) as e:                      # reserved kernel variant: refused, never silently replaced
        P.lbmk_grid_set_option(g, P.LBMK_OPT_KERNEL, P.LBMK_KERNEL_ROW)
    assert e.value.status == 6
    P.lbmk_grid_destroy(g)


def test_a_priori_subcharacteristic_check():
    """eq (2.20); Maxwell-like negative example of L393-L398: lattice speed 1 > c_s is rejected."""
    s = P.System("advection2d", params=[1.0, 0.0], tau_R=0.3, s_max=1.0)
    with pytest.raises(P.LbmkError) as e:
        P.lbmk_grid_create(s.h, 16, 16, 1, 0, 1.0, 1.0, P.LBMK_F64, 0)          # 1/lambda = 1 > 1/sqrt(3)
    assert e.value.status == 4
    g = P.lbmk_grid_create(s.h, 16, 16, 1, 0, 1.0, 2.0, P.LBMK_F64, 0)          # 0.5 <= 0.577 accepted
    P.lbmk_grid_destroy(g)
    for mk in W.BASELINE_CONFIGS.values():                                      # the lambda rule keeps all five inside
        w = mk()
        cs = math.sqrt(W.CS2[w.lattice])
        assert w.s_max / w.lam <= cs


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    s = P.System("euler2d", params=[1.4], tau_R=1.0)
    with pytest.raises(P.LbmkError) as e:
        P.Grid(s, 8, 8, 1, 0.1, 5.0)
    assert e.value.status == 3


def test_product_never_imports_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2607_05668_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "oracle/" not in text.replace("`oracle/`", "").replace("with `oracle/`", "") or f in ("__init__.py", "mms_codegen.py"), f
