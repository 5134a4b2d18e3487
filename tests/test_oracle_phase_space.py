"""Pins of the oracle's phase-space source (PAPER.md L389 names phase-space files as future work; R35
states the reading).  The expectations come from outside the new code: a source type that is pinned already
(pencil beam), exact bookkeeping of records whose fate is known without any transport, and energy conservation."""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_1101_1245_b200.inputs import (ELECTRON, PENCIL, PHASE_SPACE, PHOTON, Source, make_config,
                                         synthetic_phase_space)


def phsp_source(rec):
    return Source(PHOTON, PHASE_SPACE, 0.0, 0.0, phsp=np.asarray(rec, np.float32).reshape(-1, 8))


@pytest.mark.parametrize("particle,energy", [(PHOTON, 2.0), (ELECTRON, 6.0)])
def test_a_one_record_phase_space_is_a_pencil_beam_bit_for_bit(particle, energy):
    """The pencil beam's primaries are all (cx, cy, 0), +z, E and their transport starts at counter 1: a phase
    space holding that one record must give the same run, event for event and bit for bit."""
    w = make_config(1)
    pencil = Source(particle, PENCIL, 8.25, 8.25, energy=energy)
    rec = [[8.25, 8.25, 0.0, 0.0, 0.0, 1.0, energy, float(particle)]]
    a = oracle.run(w.density, w.material, w.voxel_cm, w.tables, pencil, 5000, seed=11)
    b = oracle.run(w.density, w.material, w.voxel_cm, w.tables, phsp_source(rec), 5000, seed=11)
    assert a.counters == b.counters
    assert np.array_equal(a.edep, b.edep)


def test_history_h_takes_record_h_mod_n_and_birth_rules():
    """Three records whose fate needs no transport: outside the phantom (escaped at birth), a photon below P_cut
    and an electron below E_cut inside known voxels (deposited where they are, R5).  With 10 histories record
    h mod 3 serves history h: 4 + 3 + 3."""
    w = make_config(1)                      # 32^3 voxels of 0.5 cm, p_cut 0.01, e_cut 0.2
    rec = [[-1.0, 3.0, 2.0, 0, 0, 1, 5.0, 0],           # outside: x < 0
           [3.2, 4.7, 6.1, 0, 0, 1, 0.0101, 0],          # photon at voxel (6, 9, 12); 0.0101 >= e_min = 0.01
           [10.0, 0.1, 15.99, 1, 0, 0, 0.15, 1]]         # electron at voxel (20, 0, 31)
    rec[1][6] = 0.01                                     # exactly e_min, below nothing: tracked ...
    tb = dataclasses.replace(w.tables, p_cut=0.02)       # ... unless the photon cutoff is raised above it
    o = oracle.run(w.density, w.material, w.voxel_cm, tb, phsp_source(rec), 10, seed=3)
    c = o.counters
    assert c["n_histories"] == 10 and c["photon_flights"] == 0 and c["ch_steps"] == 0
    assert c["e_escaped"] == pytest.approx(4 * 5.0, rel=1e-12)
    e_ph, e_el = float(np.float32(0.01)), float(np.float32(0.15))
    assert o.edep[12, 9, 6] == pytest.approx(3 * e_ph, rel=1e-12)
    assert o.edep[31, 0, 20] == pytest.approx(3 * e_el, rel=1e-12)
    assert o.edep.sum() == pytest.approx(3 * e_ph + 3 * e_el, rel=1e-12)
    assert c["e_incident"] == pytest.approx(20.0 + 3 * e_ph + 3 * e_el, rel=1e-12)


def test_mixed_phase_space_conserves_energy_and_routes_by_type():
    w = make_config(4)
    nx = w.density.shape[2]
    c0 = 0.5 * nx * w.voxel_cm
    ps = synthetic_phase_space(20_000, 17, c0, c0, 5.0, 5.0, electron_share=0.2)
    o = oracle.run(w.density, w.material, w.voxel_cm, w.tables, phsp_source(ps), 60_000, seed=5)
    c = o.counters
    tot = c["e_dep_continuous"] + c["e_dep_cutoff"] + c["e_escaped"]
    assert tot == pytest.approx(c["e_incident"], rel=1e-12)
    assert c["e_incident"] == pytest.approx(3 * ps[:, 6].astype(np.float64).sum(), rel=1e-12)
    # the electron records alone / the photon records alone: the two runs' events add up to the mixed run's
    # only in distribution (history ids differ), but each part must show its own kind of primary at work
    only_e = oracle.run(w.density, w.material, w.voxel_cm, w.tables, phsp_source(ps[ps[:, 7] == 1]), 5000, seed=5)
    only_g = oracle.run(w.density, w.material, w.voxel_cm, w.tables, phsp_source(ps[ps[:, 7] == 0]), 5000, seed=5)
    assert only_e.counters["ch_steps"] > 5 * 5000 and only_g.counters["photon_flights"] >= 5000
    ce = only_e.counters                    # photons in an electron-only run: bremsstrahlung and annihilation only
    assert ce["pushes_g"] == ce["hard_brems"] + 2 * ce["photon_pair"]


def test_phase_space_records_are_validated():
    w = make_config(1)
    ok = [8.0, 8.0, 0.0, 0, 0, 1, 2.0, 0]
    for bad in ([8.0, 8.0, 0.0, 0, 0, 1, 25.0, 0], [8.0, 8.0, 0.0, 0, 0, 1, 0.001, 1], [8.0, 8.0, 0.0, 0, 0, 1, 2.0, 2]):
        with pytest.raises(Exception):
            oracle.run(w.density, w.material, w.voxel_cm, w.tables, phsp_source([ok, bad]), 4, seed=1)
