"""Pins of the oracle's transport LOOP, where the samplers and tables are put to use (VERDICT r01 "parity
unpinned" list).  Every expectation here comes from mathematics the loop does not contain:

  * multiple-scattering strength (R12, R13): for independent, azimuthally symmetric
    deflections E[d_n | d_(n-1)] = d_(n-1) exp(-K_n), so <cos theta> after a path is exp(-int rho/lambda_1 ds),
    with 1/lambda_1 from its closed form (inputs/tables.py), in water, bone, lung and across a slab stack;
  * the alternate hinge (L139): each step multiplies <cos theta> by the mean of exp(-K) at the two energies;
  * two-body kinematics at the vertices, as pushed: momentum conservation of Compton (L65) and Moller (L88-90)
    events, the bremsstrahlung photon at theta = m/(T + m) about an unchanged electron direction (L92), pair
    electrons at opposite azimuths sharing E - 2m (L74), Sauter angles of photo-electrons (L69-70);
  * lineage: track ids of siblings, parents and all tracks of a history are pairwise distinct;
  * kinematic thresholds: no Moller event at T <= 2 K_cut, no pair event at E <= 2 m (R33).
"""
import dataclasses

import numpy as np
import pytest
from scipy import integrate, stats

import oracle
from oracle import BREMS, COMPTON, MOLLER, PAIR, PHOTO, VLOG
from paper_1101_1245_b200.inputs import ELECTRON, PENCIL, PHOTON, RECTANGLE, Source, make_config, phantoms
from paper_1101_1245_b200.inputs import materials as M
from paper_1101_1245_b200.inputs import tables as T
from paper_1101_1245_b200.inputs.tables import build_tables

M_E = 0.51099895
MATS = (M.WATER, M.BONE, M.LUNG)
f32 = lambda v: float(np.float32(v))


@pytest.fixture(scope="module")
def tables3():
    return build_tables(list(MATS))


def no_hard_events(tb, loss_scale=1.0):
    """Tables with the hard Moller / bremsstrahlung columns zeroed and the stopping power scaled."""
    tb = dataclasses.replace(tb, electron=tb.electron.copy())
    tb.electron[:, 1:3] = 0.0
    tb.electron[:, 0] *= loss_scale
    return tb


# ------------------------------------------------------------------ multiple-scattering strength
@pytest.mark.parametrize("m,rho,T0,es", [(0, 1.0, 2.0, 0.04), (1, 1.85, 3.0, 0.04), (2, 0.26, 1.0, 0.04), (0, 0.5, 6.0, 0.4)])
def test_ms_strength_in_a_uniform_medium(m, rho, T0, es, tables3):
    """One voxel far larger than the path, no energy loss, no hard events: every step has length e_s-max, so
    after n steps <cos theta> = exp(-n e_s rho / lambda_1(T)) exactly (column, density and step length)."""
    tb = no_hard_events(tables3, 1e-9)
    h, es, n_steps, n = 1000.0, f32(es), 30, 150_000
    dens, mat = phantoms.homogeneous(1, 1, 1, rho, m)
    src = Source(ELECTRON, PENCIL, 500.0, 500.0, energy=T0)
    end, path = oracle.run_endstate(dens, mat, h, tb, src, n, seed=61, options=oracle.Options(es_max_cm=es),
                                    max_steps=n_steps)
    steps = end[:, 7]
    full = steps == n_steps                    # the others were back-scattered out of the entrance face (z = 0)
    assert full.mean() > 0.9 and np.mean(np.isclose(path[:, m], n_steps * es, rtol=1e-12)) > 0.9
    assert np.all(path[:, m] <= steps * es * (1 + 1e-12))      # (a step towards the entrance face ends there)
    assert np.allclose(end[:, 6], T0, rtol=1e-6)
    k_cm = rho * float(T.inv_lambda1_mass(MATS[m], T0))         # rho / lambda_1, from the definition
    K = n_steps * es * k_cm
    assert 0.3 < K < 2.5
    cos = end[:, 5]                                        # the beam starts along +z
    # exact, whatever happens at the entrance face: d_n exp(sum K) is a martingale, stopped at the track's end
    mart = cos * np.exp(k_cm * path[:, m])
    assert abs(mart.mean() - 1.0) < 3.5 * mart.std() / np.sqrt(n) + 3e-4 * K
    # and in the paper's words, for the tracks that made all their steps inside (the others carry at most
    # their share of the mean)
    lost = 1.0 - full.mean()
    assert abs(cos.mean() - np.exp(-K)) < 3.5 * cos.std() / np.sqrt(n) + 3e-4 * K + 2 * lost
    # no net sideways drift of the direction
    assert abs(end[:, 3].mean()) < 4 * end[:, 3].std() / np.sqrt(n)
    assert abs(end[:, 4].mean()) < 4 * end[:, 4].std() / np.sqrt(n)


def test_ms_strength_across_a_slab_stack(tables3):
    """Water / bone / lung / water slabs (config 4's stack), cubic voxels, no energy loss, no hard events.
    Step lengths now depend on the direction (d_vox), but M_n = d_n exp(+sum_i K_i) is a martingale, so at the
    (bounded) end of the track E[cos theta_end exp(int rho/lambda_1 ds)] = 1 exactly; the integral is taken over
    the path the oracle reports per material, with rho and 1/lambda_1 from their definitions."""
    tb = no_hard_events(tables3, 1e-9)
    h, T0, n = 0.25, 10.0, 120_000
    dens, mat = phantoms.z_slabs(96, 96, 64, [(12, 1.0, 0), (8, 1.85, 1), (28, 0.26, 2), (None, 1.0, 0)])
    src = Source(ELECTRON, PENCIL, 12.125, 12.125, energy=T0)
    end, path = oracle.run_endstate(dens, mat, h, tb, src, n, seed=62, max_steps=400)
    rho = np.array([1.0, 1.85, 0.26])
    inv_l1 = np.array([float(T.inv_lambda1_mass(mm, T0)) for mm in MATS])
    K = path @ (rho * inv_l1)
    # most tracks cross all slabs (thicknesses 3 + 4, 2, 7 cm) and leave through the far face; the shape's
    # single-scattering tail sends the others out sideways or back: the martingale covers them all
    assert np.mean(end[:, 2] >= 16.0) > 0.5 and np.mean(end[:, 7] >= 400) < 0.01
    far = end[:, 2] >= 16.0
    assert np.all(path[far] >= [6.5, 1.5, 6.5])    # (a step is booked on the material it starts in)
    assert path[far].mean(axis=0) == pytest.approx([7.0, 2.0, 7.0], rel=0.25)     # detours included
    assert 0.4 < K.mean() < 1.2
    mart = end[:, 5] * np.exp(K)
    assert abs(mart.mean() - 1.0) < 3.5 * mart.std() / np.sqrt(n) + 3e-4
    # a dropped density, a wrong column or a forgotten step length breaks it far beyond the noise
    for wrong in (path @ inv_l1, path @ rho * inv_l1[0], 0.5 * K):
        bad = end[:, 5] * np.exp(wrong)
        assert abs(bad.mean() - 1.0) > 10 * bad.std() / np.sqrt(n)


def test_alternate_hinge_uses_the_energy_before_or_after_the_loss(tables3):
    """L139 / R12: with real energy loss each step scatters with the strength at T or at T - dE, probability
    1/2 each, so <cos theta_n> = prod_k (exp(-K_k(T_k)) + exp(-K_k(T_k+1)))/2.  The energies T_k and step
    lengths are read off the oracle step by step (they are pinned by the CSDA tests)."""
    tb = no_hard_events(tables3)
    h, T0, n, n_steps = 1000.0, 2.0, 150_000, 5
    dens, mat = phantoms.homogeneous(1, 1, 1, 1.0, 0)
    src = Source(ELECTRON, PENCIL, 500.0, 500.0, energy=T0)
    Ts, ss = [T0], []
    for k in range(1, n_steps + 1):
        e, p = oracle.run_endstate(dens, mat, h, tb, src, 2, seed=63, max_steps=k)
        Ts.append(e[0, 6])
        ss.append(p[0, 0] - sum(ss))
    assert Ts[-1] < 0.6 * T0 and all(0.05 < s <= 0.5 for s in ss)
    end, path = oracle.run_endstate(dens, mat, h, tb, src, n, seed=63, max_steps=n_steps)
    il1 = lambda t: T.inv_lambda1_mass(M.WATER, t)
    steps = end[:, 7].astype(int)
    assert np.mean(steps == n_steps) > 0.8
    # every track's product of step factors; a track that left through the entrance face made a shorter last
    # step, whose length and end energy are in its end state
    done = np.concatenate([[0.0], np.cumsum(ss)])
    fac = {"both": np.ones(n), "before": np.ones(n), "after": np.ones(n)}
    for k in range(n_steps):
        on = steps > k
        last_short = on & (steps == k + 1) & (steps < n_steps)
        s_k = np.where(last_short, path[:, 0] - done[k], ss[k])
        T_after = np.where(last_short, end[:, 6], Ts[k + 1])
        a, b = np.exp(-s_k * il1(Ts[k])), np.exp(-s_k * il1(np.maximum(T_after, 1e-3)))
        for name, f in (("both", 0.5 * (a + b)), ("before", a), ("after", b)):
            fac[name] = np.where(on, fac[name] * f, fac[name])
    cos = end[:, 5]
    mart = cos / fac["both"]
    assert abs(mart.mean() - 1.0) < 3.5 * mart.std() / np.sqrt(n) + 2e-3
    for name in ("before", "after"):                      # the test can tell the alternatives apart
        bad = cos / fac[name]
        assert abs(bad.mean() - 1.0) > 10 * bad.std() / np.sqrt(n)
    full = steps == n_steps
    assert abs(cos[full].mean() - fac["both"][full][0]) < 0.05 * fac["both"][full][0] + 2 * (1 - full.mean())


# ------------------------------------------------------------------ vertices, as pushed
@pytest.fixture(scope="module")
def vertices_15MeV():
    """Config 3 (15 MeV photons in water): Compton, pair, Moller and bremsstrahlung vertices in quantity."""
    w = make_config(3)
    rows, c = oracle.run_vertices(w.density, w.material, w.voxel_cm, w.tables, w.source, 60_000, seed=71)
    assert rows.shape[0] == c["pushes_e"] + c["pushes_g"] > 100_000
    return rows, w


def unit(v):
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def momentum(T):
    return np.sqrt(T * (T + 2 * M_E))


def azimuth_about(d0, d):
    """Azimuth of d about d0 in a frame that depends on d0 only."""
    ref = np.where(np.abs(d0[:, 2:3]) < 0.9, np.array([[0.0, 0.0, 1.0]]), np.array([[1.0, 0.0, 0.0]]))
    e1 = unit(np.cross(d0, ref))
    e2 = np.cross(d0, e1)
    return np.arctan2((d * e2).sum(1), (d * e1).sum(1))


def test_compton_recoil_conserves_momentum(vertices_15MeV):
    """L65: free electron at rest, so E d = E' d' + p_e d_e with p_e = sqrt(T (T + 2m)), T = E - E'."""
    rows, _ = vertices_15MeV
    r = rows[rows[:, VLOG["kind"]] == COMPTON]
    assert len(r) > 20_000 and np.all(r[:, VLOG["child_type"]] == 1)
    E0, E1, Te = r[:, VLOG["E0"]], r[:, VLOG["E1"]], r[:, VLOG["child_E"]]
    np.testing.assert_allclose(Te, E0 - E1, rtol=1e-14)
    lhs = E0[:, None] * r[:, VLOG["d0"]]
    rhs = E1[:, None] * r[:, VLOG["d1"]] + momentum(Te)[:, None] * r[:, VLOG["child_d"]]
    assert np.abs(lhs - rhs).max() <= 1e-12 * E0.max()
    np.testing.assert_allclose(np.linalg.norm(r[:, VLOG["child_d"]], axis=1), 1.0, rtol=1e-14)
    # and the scattered photon obeys the Compton relation in situ
    cos_g = (r[:, VLOG["d0"]] * r[:, VLOG["d1"]]).sum(1)
    np.testing.assert_allclose(E1, E0 / (1 + E0 / M_E * (1 - cos_g)), rtol=1e-9)


def test_moller_vertices_conserve_energy_and_momentum(vertices_15MeV):
    """L88-90: both outgoing electrons, as the loop emits them (angles, opposite azimuths, who gets which)."""
    rows, w = vertices_15MeV
    r = rows[rows[:, VLOG["kind"]] == MOLLER]
    assert len(r) > 30_000 and np.all(r[:, VLOG["child_type"]] == 1)
    T0, T1, W = r[:, VLOG["E0"]], r[:, VLOG["E1"]], r[:, VLOG["child_E"]]
    np.testing.assert_allclose(T1 + W, T0, rtol=1e-14)
    assert np.all(W >= w.tables.e_cut * (1 - 1e-12)) and np.all(W <= 0.5 * T0 * (1 + 1e-12))
    assert np.all(T0 > 2 * f32(w.tables.e_cut))                                  # R33
    lhs = momentum(T0)[:, None] * r[:, VLOG["d0"]]
    rhs = momentum(T1)[:, None] * r[:, VLOG["d1"]] + momentum(W)[:, None] * r[:, VLOG["child_d"]]
    assert np.abs(lhs - rhs).max() <= 1e-9 * momentum(T0).max()
    phi = azimuth_about(r[:, VLOG["d0"]], r[:, VLOG["child_d"]])
    assert stats.kstest((phi + np.pi) / (2 * np.pi), "uniform").pvalue > 0.01


def test_bremsstrahlung_vertices(vertices_15MeV):
    """L92: "the direction of the electron is unchanged", photon at polar angle m/E about it, E the electron's
    total energy (R14); the photon energy comes off the electron."""
    rows, w = vertices_15MeV
    r = rows[rows[:, VLOG["kind"]] == BREMS]
    assert len(r) > 15_000 and np.all(r[:, VLOG["child_type"]] == 0)
    T0, T1, k = r[:, VLOG["E0"]], r[:, VLOG["E1"]], r[:, VLOG["child_E"]]
    np.testing.assert_allclose(T1 + k, T0, rtol=1e-14)
    assert np.all(k >= f32(w.tables.p_cut) * (1 - 1e-12)) and np.all(k <= T0)
    assert np.array_equal(r[:, VLOG["d0"]], r[:, VLOG["d1"]])
    cos_t = (r[:, VLOG["d0"]] * r[:, VLOG["child_d"]]).sum(1)
    sin_t = np.linalg.norm(np.cross(r[:, VLOG["d0"]], r[:, VLOG["child_d"]]), axis=1)
    np.testing.assert_allclose(np.arctan2(sin_t, cos_t), M_E / (T0 + M_E), rtol=1e-9)
    phi = azimuth_about(r[:, VLOG["d0"]], r[:, VLOG["child_d"]])
    assert stats.kstest((phi + np.pi) / (2 * np.pi), "uniform").pvalue > 0.01


def vertex_key(r):
    return r[:, VLOG["hist"]] * 2.0**40 + r[:, VLOG["parent_track"]] * 2.0**8 + r[:, VLOG["parent_ctr"]]


def test_pair_vertices(vertices_15MeV):
    """L74: two electrons share E - 2m, opposite azimuths, polar density (1 - beta cos)^-2; R6: the rest energy
    leaves as two back-to-back isotropic 0.511 MeV photons."""
    rows, w = vertices_15MeV
    r = rows[rows[:, VLOG["kind"]] == PAIR]
    assert np.all(r[:, VLOG["E0"]] > 2 * M_E)                                    # R33
    g = r[r[:, VLOG["child_type"]] == 0]
    e = r[r[:, VLOG["child_type"]] == 1]
    # photons: pushed in pairs, one after the other
    assert len(g) % 2 == 0 and len(g) > 15_000
    ga, gb = g[0::2], g[1::2]
    assert np.array_equal(vertex_key(ga), vertex_key(gb))
    assert np.all(g[:, VLOG["child_E"]] == M_E)
    np.testing.assert_allclose(ga[:, VLOG["child_d"]], -gb[:, VLOG["child_d"]], atol=1e-15)
    assert stats.kstest((ga[:, VLOG["child_d"]][:, 2] + 1) / 2, "uniform").pvalue > 0.01
    assert stats.kstest((np.arctan2(ga[:, 16], ga[:, 15]) + np.pi) / (2 * np.pi), "uniform").pvalue > 0.01
    # electrons: vertices where both were above the cutoff
    key = vertex_key(e)
    same = key[1:] == key[:-1]
    a, b = e[:-1][same], e[1:][same]
    assert len(a) > 8_000
    E0 = a[:, VLOG["E0"]]
    np.testing.assert_allclose(a[:, VLOG["child_E"]] + b[:, VLOG["child_E"]], E0 - 2 * M_E, rtol=1e-12)
    d0 = a[:, VLOG["d0"]]
    ta = a[:, VLOG["child_d"]] - (a[:, VLOG["child_d"]] * d0).sum(1, keepdims=True) * d0
    tb_ = b[:, VLOG["child_d"]] - (b[:, VLOG["child_d"]] * d0).sum(1, keepdims=True) * d0
    ok = (np.linalg.norm(ta, axis=1) > 1e-6) & (np.linalg.norm(tb_, axis=1) > 1e-6)
    assert np.allclose((unit(ta[ok]) * unit(tb_[ok])).sum(1), -1.0, atol=1e-6)   # opposite azimuths
    for x in (a, b):
        Tk = x[:, VLOG["child_E"]]
        beta = momentum(Tk) / (Tk + M_E)
        c = (x[:, VLOG["child_d"]] * d0).sum(1)
        cdf = (1 / (1 - beta * c) - 1 / (1 + beta)) / (1 / (1 - beta) - 1 / (1 + beta))
        assert stats.kstest(np.clip(cdf, 0, 1), "uniform").pvalue > 0.01
    # the split is uniform (first electron of a vertex where both are tracked: uniform on the allowed range)
    Ts = E0 - 2 * M_E
    lo = f32(w.tables.e_cut) / Ts
    u = (a[:, VLOG["child_E"]] / Ts - lo) / (1 - 2 * lo)
    assert stats.kstest(u, "uniform").pvalue > 0.01


def test_photoelectron_vertices(tables3):
    """L67-72: T = E_phot, Sauter polar angle, uniform azimuth; 0.3 MeV photons on bone, first interactions."""
    E, n = 0.3, 400_000
    dens, mat = phantoms.homogeneous(8, 8, 40, 1.85, 1)
    src = Source(PHOTON, PENCIL, 2.125, 2.125, energy=E)
    rows, c = oracle.run_vertices(dens, mat, 0.5, tables3, src, n, seed=72)
    r = rows[(rows[:, VLOG["kind"]] == PHOTO) & (rows[:, VLOG["parent_track"]] == 0) & (rows[:, VLOG["E0"]] == f32(E))]
    assert len(r) > 1500
    assert np.all(r[:, VLOG["child_E"]] == r[:, VLOG["E0"]]) and np.all(r[:, VLOG["E1"]] == 0.0)
    assert np.all(r[:, VLOG["d0"]] == [0.0, 0.0, 1.0])
    nu = 1.0 - r[:, VLOG["child_d"]][:, 2]
    E = f32(E)
    gam = 1 + E / M_E
    beta = np.sqrt(E * (E + 2 * M_E)) / (E + M_E)
    A, B = 1 / beta - 1, 0.5 * beta * gam * (gam - 1) * (gam - 2)
    pdf = lambda v: (2 - v) * (1 / (A + v) + B) * v / (A + v) ** 3
    norm = integrate.quad(pdf, 0, 2)[0]
    cdf = np.vectorize(lambda v: integrate.quad(pdf, 0, v)[0] / norm)
    assert stats.kstest(nu, cdf).pvalue > 0.01
    phi = np.arctan2(r[:, 16], r[:, 15])
    assert stats.kstest((phi + np.pi) / (2 * np.pi), "uniform").pvalue > 0.01


def test_lineage_gives_every_track_of_a_history_its_own_id(vertices_15MeV):
    """children take distinct words of the lineage block; a shared id would correlate tracks."""
    rows, _ = vertices_15MeV
    hist = rows[:, VLOG["hist"]].astype(np.int64)
    child = rows[:, VLOG["child_track"]].astype(np.int64)
    parent = rows[:, VLOG["parent_track"]].astype(np.int64)
    assert len(rows) > 100_000
    assert np.all(child != parent) and np.all(child != 0)            # track 0 is the primary
    # within a history no two tracks share an id (chance collisions: ~n^2 / 2^33 per history, ~1e-5 in all)
    key = hist * (1 << 32) + child
    assert len(np.unique(key)) == len(key)
    # siblings of one vertex (pair: up to four) are distinct in particular, and ids are spread over 32 bits
    assert stats.kstest(child / 2.0**32, "uniform").pvalue > 0.001
    # a parent's later vertices get new ids although its track id stays: the draw counter enters
    vk = vertex_key(rows)
    assert len(np.unique(vk)) > 0.6 * len(rows)


# ------------------------------------------------------------------ kinematic thresholds (R33)
def test_no_moller_event_below_twice_the_cutoff(water_tables):
    """The Moller column is zero at the node below 2 K_cut and positive at the node above it, so its
    interpolant is positive just below the threshold, where eps in [K_cut/T, 1/2] is empty."""
    tb = water_tables
    lnE = np.linspace(np.log(tb.e_min), np.log(tb.e_max), tb.n_energy)
    T0 = 0.3995
    assert np.interp(np.log(T0), lnE, tb.electron[0, 1].astype(np.float64)) > 0          # the trap is there
    dens, mat = phantoms.homogeneous(4, 4, 4, 1.0, 0)
    src = Source(ELECTRON, PENCIL, 0.5, 0.5, energy=T0)
    # inflate the hard-event rate so that the candidates are many: all must be fictitious or bremsstrahlung
    r = oracle.run(dens, mat, 0.25, tb, src, 300_000, seed=81, options=oracle.Options(majorant_scale=200.0))
    assert r.counters["hard_fict"] > 100_000
    assert r.counters["hard_moller"] == 0
    ok = oracle.run(dens, mat, 0.25, tb, dataclasses.replace(src, energy=0.45), 100_000, seed=81)
    assert ok.counters["hard_moller"] > 0


def test_coarse_tables_cannot_produce_negative_deposits():
    """With few energy nodes the interpolated pair and Moller columns reach far below their thresholds
    (ADVICE r01): no pair event below 2 m, no negative energy anywhere."""
    tb = build_tables([M.WATER], n_energy=20)
    lnE = np.linspace(np.log(tb.e_min), np.log(tb.e_max), tb.n_energy)
    assert np.interp(np.log(1.0), lnE, tb.photon[0, 2].astype(np.float64)) > 0           # the trap is there
    dens, mat = phantoms.homogeneous(16, 16, 64, 1.0, 0)
    src = Source(PHOTON, PENCIL, 2.125, 2.125, energy=1.0)
    r = oracle.run(dens, mat, 0.25, tb, src, 200_000, seed=82)
    assert r.counters["photon_pair"] == 0 and r.counters["photon_compton"] > 100_000
    assert np.all(r.edep >= 0.0)
    c = r.counters
    assert abs((c["e_dep_continuous"] + c["e_dep_cutoff"] + c["e_escaped"]) / c["e_incident"] - 1) < 1e-12
    src = Source(ELECTRON, PENCIL, 2.125, 2.125, energy=0.39)
    r = oracle.run(dens, mat, 0.25, tb, src, 100_000, seed=83, options=oracle.Options(majorant_scale=50.0))
    assert r.counters["hard_moller"] == 0 and np.all(r.edep >= 0.0)
