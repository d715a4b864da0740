"""Host-side logic of libqss (no GPU): ABI surface, mechanism validation, SCC ordering of the QSS groups
(App. B), the branch-free exp, and the cell sharding used at N > 1."""
import ctypes as ct
import os
import re
import subprocess
import sys

import numpy as np
import pytest

import paper_2405_05974_b200 as qss
import qss_synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_symbol_of_the_header():
    hdr = open(os.path.join(ROOT, "include", "qss.h")).read()
    declared = sorted(set(re.findall(r"\b(qss_[a-z0-9_]+)\s*\(", hdr)))
    assert set(declared) == set(qss.EXPORTS), (declared, qss.EXPORTS)
    L = qss.lib()
    for name in declared:
        assert getattr(L, name) is not None


def test_no_cpu_fallback_create_fails_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(qss.QssError) as e:
        qss.QssMech(qss_synth.toy1(), 0)
    assert e.value.code == -6            # QSS_E_CUDA


@pytest.mark.parametrize("cfg,gmax", [(1, 3), (2, 4), (3, 6)])
def test_group_sizes_of_the_configs(cfg, gmax):
    mech = qss_synth.config_mechanism(cfg)
    ng, order, grp = qss.validate(mech)
    assert sorted(order.tolist()) == list(range(mech.n_qss))
    sizes = np.bincount(grp, minlength=ng)
    assert sizes.max() == gmax and sizes.sum() == mech.n_qss


def _edges(mech):
    """QSS digraph: n -> m iff an enabled direction consumes QSS n and produces QSS m."""
    N = mech.n_nqss
    E = set()
    for j in range(mech.n_reac):
        R = [int(s) for s in mech.reac_sp[mech.reac_ptr[j]:mech.reac_ptr[j + 1]] if s >= N]
        P = [int(s) for s in mech.prod_sp[mech.prod_ptr[j]:mech.prod_ptr[j + 1]] if s >= N]
        if mech.dir_mask[j] & 1:
            E |= {(n - N, m - N) for n in R for m in P if n != m}
        if mech.dir_mask[j] & 2:
            E |= {(n - N, m - N) for n in P for m in R if n != m}
    return E


@pytest.mark.parametrize("make", [qss_synth.toy_dag, lambda: qss_synth.config_mechanism(2), lambda: qss_synth.config_mechanism(3)])
def test_groups_are_the_sccs_in_topological_order(make):
    mech = make()
    ng, order, grp = qss.validate(mech)
    g_of = {int(q): int(g) for q, g in zip(order, grp)}
    E = _edges(mech)
    # solve order respects every edge: the producer side n of n -> m is solved no later than m
    assert all(g_of[n] <= g_of[m] for n, m in E)
    # two species share a group iff they reach each other (brute-force transitive closure)
    nq = mech.n_qss
    reach = np.eye(nq, dtype=bool)
    for n, m in E:
        reach[n, m] = True
    for k in range(nq):
        reach |= reach[:, k:k + 1] & reach[k:k + 1, :]
    for a in range(nq):
        for b in range(nq):
            assert (g_of[a] == g_of[b]) == bool(reach[a, b] and reach[b, a])


def _with(mech, **kw):
    import dataclasses
    return dataclasses.replace(mech, **kw)


def test_validation_errors():
    m = qss_synth.toy2()                                   # A <=> Q1, Q1 <=> Q2, Q2 <=> B ; species A B Q1 Q2
    # quadratic coupling: 2 Q1 on the reactant side of an enabled direction
    bad = _with(m, reac_nu=np.array([1, 2, 1], dtype=np.int32))
    with pytest.raises(qss.QssError) as e:
        qss.validate(bad)
    assert e.value.code == -2
    # the same side only produced (reverse disabled... forward consumes Q1 twice) -> still quadratic; disable forward: fan-out
    bad2 = _with(bad, dir_mask=np.array([3, 2, 3], dtype=np.uint8))
    with pytest.raises(qss.QssError) as e:
        qss.validate(bad2)
    assert e.value.code == -3
    # no sink: Q2 can only be produced, never consumed towards a transported species
    bad3 = _with(m, dir_mask=np.array([3, 1, 2], dtype=np.uint8))
    with pytest.raises(qss.QssError) as e:
        qss.validate(bad3)
    assert e.value.code == -4
    # unsupported reaction type, bad species index
    with pytest.raises(qss.QssError) as e:
        qss.validate(_with(m, rtype=np.array([0, 7, 0], dtype=np.int32)))
    assert e.value.code == -5
    with pytest.raises(qss.QssError) as e:
        qss.validate(_with(m, reac_sp=np.array([0, 2, 9], dtype=np.int32)))
    assert e.value.code == -1


def test_strict_element_balance_and_parameter_validation():
    """strict_balance (QSS_E_UNBALANCED): every reaction must conserve every element; duplicate third-body
    efficiencies and unusable Troe temperatures are rejected; CHEMKIN placeholders are accepted."""
    for make in (qss_synth.toy1, qss_synth.toy_dag, lambda: qss_synth.config_mechanism(1), lambda: qss_synth.config_mechanism(2)):
        qss.validate(make(), strict_balance=True)
    m = qss_synth.config_mechanism(1)
    comp = m.comp.copy(); comp[int(m.reac_sp[0]), 0] += 1
    bad = _with(m, comp=comp)
    qss.validate(bad)                                      # not strict: the compositions are not looked at
    with pytest.raises(qss.QssError) as e:
        qss.validate(bad, strict_balance=True)
    assert e.value.code == -7
    m2 = qss_synth.config_mechanism(2)
    j = int(np.flatnonzero(m2.rtype == 2)[0])
    for k, val in ((1, 0.0), (2, -5.0), (0, float("nan")), (3, float("inf"))):
        troe = m2.troe.copy(); troe[j, k] = val
        with pytest.raises(qss.QssError) as e:
            qss.validate(_with(m2, troe=troe))
        assert e.value.code == -1
    troe = m2.troe.copy(); troe[j] = (0.4, 1e-30, 1e30, 1e30)
    qss.validate(_with(m2, troe=troe))
    jt = int(np.flatnonzero(np.diff(m2.eff_ptr) >= 2)[0])
    eff_sp = m2.eff_sp.copy(); eff_sp[m2.eff_ptr[jt] + 1] = eff_sp[m2.eff_ptr[jt]]
    with pytest.raises(qss.QssError) as e:
        qss.validate(_with(m2, eff_sp=eff_sp))
    assert e.value.code == -1


def test_compiled_images_are_cached_on_disk(tmp_path, monkeypatch):
    """qss_jit.cpp: the run-time compiled image of a mechanism is written to $QSS_CACHE_DIR, keyed by a hash of every source;
    a second process-independent compilation of the same mechanism finds it (checked through the file set, no GPU needed)."""
    monkeypatch.setenv("QSS_CACHE_DIR", str(tmp_path / "cache"))
    n1 = qss.specialise_check(qss_synth.toy2(), (10, 0))
    files = sorted(os.listdir(tmp_path / "cache"))
    assert len(files) == 1 and files[0].endswith(".cubin") and os.path.getsize(tmp_path / "cache" / files[0]) == n1
    qss.specialise_check(qss_synth.toy3(), (10, 0))
    assert len(os.listdir(tmp_path / "cache")) == 2
    monkeypatch.setenv("QSS_CACHE", "0")
    monkeypatch.setenv("QSS_CACHE_DIR", str(tmp_path / "off"))
    qss.specialise_check(qss_synth.toy1(), (10, 0))
    assert not os.path.exists(tmp_path / "off")


def test_specialised_jacobian_kernel_compiles_without_a_gpu():
    """Run-time specialisation, host side: the generated source of a mechanism's Jacobian columns compiles with NVRTC for
    sm_100a (no device needed); a mechanism outside kernel variant 1 has nothing to specialise."""
    for mech in (qss_synth.toy_dag(), qss_synth.config_mechanism(1)):
        assert qss.specialise_check(mech, (10, 0)) > 10000
    # species with their own NASA-7 mid temperatures: the image carries the range-correction path of the rate tasks (G_HAS_CORR)
    import dataclasses
    mech = qss_synth.config_mechanism(1)
    nasa_T = mech.nasa_T.copy()
    nasa_T[:, 1] = np.linspace(950.0, 1400.0, nasa_T.shape[0])
    assert qss.specialise_check(dataclasses.replace(mech, nasa_T=nasa_T), (10, 0)) > qss.specialise_check(mech, (10, 0))
    with pytest.raises(qss.QssError) as ei:
        qss.specialise_check(qss_synth.config_mechanism(5), (10, 0))
    assert ei.value.code == -5


def test_branch_free_exp_against_float128(tmp_path):
    """csrc/qss_math.h compiled for the host: <= 1.5 ulp against libquadmath over the whole finite range."""
    src = tmp_path / "t.cpp"
    src.write_text(r'''
#include "qss_math.h"
#include <cstdio>
#include <random>
#include <quadmath.h>
int main() {
  std::mt19937_64 g(1); double worst = 0, worst_e = 0, worst_t = 0;
  double tab[64]; for (int j = 0; j < 64; ++j) tab[j] = (double)exp2l((long double)j / 64.0L);      // as csrc/qss_gen3.cpp writes it
  std::uniform_real_distribution<double> u(-745.0, 709.0), s(-1.0, 1.0);
  for (int i = 0; i < 2000000; ++i) {
    double x = (i & 1) ? u(g) : s(g), a = qss_exp(x), b = qss_exp_e(x); __float128 r = expq((__float128)x); double rd = (double)r;
    if (rd == 0 || std::isinf(rd)) continue;
    double ulp = std::fabs(std::nextafter(rd, INFINITY) - rd), e = (double)fabsq((__float128)a - r) / ulp;
    if (e > worst) worst = e;
    e = (double)fabsq((__float128)b - r) / ulp;
    if (e > worst_e) worst_e = e;
    e = (double)fabsq((__float128)qss_exp_tab(x, (const double *)tab) - r) / ulp;
    if (e > worst_t) worst_t = e;
  }
  const int tab_ok = qss_exp_tab(0.0, (const double *)tab) == 1.0 && qss_exp_tab(-1000.0, (const double *)tab) == 0.0 && std::isinf(qss_exp_tab(1000.0, (const double *)tab)) &&
                     qss_exp_tab(-746.0, (const double *)tab) == 0.0 && std::isinf(qss_exp_tab(710.0, (const double *)tab));
  // saturating form for placeholder arguments (fall-off temperatures 1e-30 / 1e30): 0, 1 and inf like the library function
  const int sat = qss_exp_sat(-1.4e33) == 0.0 && qss_exp_sat(-1e27) == 0.0 && qss_exp_sat(-2e9) == 0.0 && qss_exp_sat(-1.4e-27) == 1.0 &&
                  std::isinf(qss_exp_sat(1e12)) && qss_exp_sat(-INFINITY) == 0.0 && qss_exp_sat(0.5) == qss_exp(0.5);
  printf("%.4f %d %d %d %.4f %d %.4f %d\n", worst, qss_exp(0.0) == 1.0, qss_exp(-1000.0) == 0.0, std::isinf(qss_exp(1000.0)), worst_e, sat, worst_t, tab_ok);
}''')
    exe = tmp_path / "t"
    subprocess.run(["g++", "-O2", "-ffp-contract=off", "-I", os.path.join(ROOT, "paper_2405_05974_b200", "csrc"), "-o", str(exe),
                    str(src), "-lquadmath"], check=True)
    worst, one, zero, inf, worst_e, sat, worst_t, tab_ok = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()
    assert float(worst) <= 1.5 and one == "1" and zero == "1" and inf == "1"
    assert float(worst_e) <= 2.5, worst_e            # Estrin form of the polynomial (kernel variant 3)
    assert sat == "1"
    assert float(worst_t) <= 1.5 and tab_ok == "1", (worst_t, tab_ok)            # table form (kernel variant 3's rate phase)


def test_cell_ranges_tile_the_cells():
    from paper_2405_05974_b200.shard import cell_range
    for n in (0, 1, 31, 32, 33, 4096, 2 ** 20, 2 ** 20 + 5):
        for world in (1, 2, 3, 8):
            r = [cell_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            assert all(b % 32 == 0 or b == n for b, _ in r)
            sizes = [e - b for b, e in r]
            assert max(sizes) - min(sizes) < 64 or n < 32 * world


def _gloo_worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2405_05974_b200.shard import cell_range, max_over_ranks
    b, e = cell_range(1000, rank, world)
    t = max_over_ranks(1.0 + rank, dist)
    q.put((rank, b, e, t))
    dist.destroy_process_group()


def test_two_rank_sharding_and_timing_reduction_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 500
    ps = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in ps]
    out = sorted(q.get(timeout=120) for _ in ps)
    [p.join(60) for p in ps]
    assert out[0][1:3] == (0, 512) and out[1][1:3] == (512, 1000)
    assert out[0][3] == 2.0 and out[1][3] == 2.0          # max over ranks


@pytest.mark.parametrize("name", ["toy3", "toy_dag", "cfg1", "cfg2"])
def test_structural_jacobian_pattern_against_the_oracle(name):
    """NEXT-3 (Table 4): qss_mech_jac_pattern is host logic; every numerically non-zero entry of the oracle's Jacobian (any
    of 40 random states, the paper's sampling) lies inside the structural pattern of the same mode, and on the generic synthetic
    mechanisms the two coincide; the chain term only ever adds entries (exact >= constant-QSS >= zero-QSS)."""
    import oracle
    mech = qss_synth.config_mechanism(int(name[3])) if name.startswith("cfg") else getattr(qss_synth, name)()
    N = mech.n_nqss; n = 40
    rng = np.random.default_rng(1)
    C = np.ascontiguousarray(rng.uniform(1e-4, 1.0, size=(N, n))); T = rng.uniform(300.0, 1300.0, size=n)
    om = oracle.OracleMech(mech)
    pats = []
    for mode, omode in ((0, oracle.EXPLICIT_F64), (1, oracle.JAC_CONST_QSS), (2, oracle.JAC_ZERO_QSS)):
        pat = qss.jac_pattern(mech, mode).astype(bool)
        with np.errstate(all="ignore"):
            num = (oracle.evaluate(om, C, T, mode=omode)["jac"] != 0).any(2)
        assert not (num & ~pat).any(), (name, mode)
        if name.startswith("cfg"):
            assert np.array_equal(num, pat), (name, mode)
        pats.append(pat)
        print("%s mode %d: fill of the N x N block %.3f" % (name, mode, pat[:, :N].mean()))
    assert not (pats[1] & ~pats[0]).any() and not (pats[2] & ~pats[1]).any()
