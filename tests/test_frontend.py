"""File front-end: the seven .in formats, the append-mode .out files, the driver input
file.  Host logic only; the simulation behind run_folder is the oracle here (tests may use it) and the
CUDA library in tests/test_gpu_transport.py."""
import os

import numpy as np
import pytest

from paper_1705_01387_b200 import frontend as F
from workloads import lattices as L


def _same(a, b):
    if a is None or b is None:
        return a is None and b is None
    return np.asarray(a).tobytes() == np.asarray(b).tobytes()


@pytest.mark.parametrize("model", [
    L.square(6, 5, W=2.0, seed=1),                                               # no hopping.in (all -1)
    L.with_bond_disorder(L.graphene(4, 3, vacancy_fraction=0.2, vacancy_seed=3), 0.3, 5),   # real hoppings, ragged rows
    L.square_peierls(6, 4, flux_quanta=1, W=1.0, seed=2),                        # complex hoppings
    L.chain(7, periodic=False),                                                  # no potential.in
], ids=["default_hop", "real_hop_ragged", "complex_hop", "no_potential"])
def test_folder_round_trip_is_bit_exact(tmp_path, model):
    E = np.linspace(-3.0, 3.0, 7)
    dts = np.array([0.1, 0.25, 1.0 / 3.0])
    F.write_folder(str(tmp_path), model, E, dts, {"calculate_msd": True, "number_of_moments": 64})
    assert os.path.exists(tmp_path / "hopping.in") == (model.hop_re is not None)
    assert os.path.exists(tmp_path / "potential.in") == (model.onsite is not None)
    got, para, E2, dts2 = F.read_folder(str(tmp_path))
    assert (got.N, got.K) == (model.N, model.K)
    assert _same(got.nbr_count, model.nbr_count)
    valid = (np.arange(model.K)[None, :] < model.nbr_count[:, None]).reshape(-1)
    assert np.array_equal(got.nbr_index[valid], model.nbr_index[valid])          # 0-based, as written
    for a, b in ((got.hop_re, model.hop_re), (got.hop_im, model.hop_im)):
        assert (a is None) == (b is None)
        if a is not None:
            assert _same(a[valid], b[valid])                                     # repr() round-trips doubles exactly
    assert _same(got.onsite, model.onsite) and _same(got.x, model.x)
    assert (got.box_length, got.volume, got.energy_scale) == (model.box_length, model.volume, model.energy_scale)
    assert _same(E2, E) and _same(dts2, dts)
    assert para["calculate_msd"] and not para["calculate_vac"] and para["number_of_moments"] == 64
    assert para["number_of_random_vectors"] == 1                                 # default


def test_para_defaults_blank_lines_and_errors(tmp_path):
    p = tmp_path / "para.in"
    assert F.read_para(str(p)) == F.DEFAULTS                                     # file absent: all defaults
    p.write_text("\n\ncalculate_vac\n\nnumber_of_random_vectors 3\n   \nenergy_max 6.1\n")
    para = F.read_para(str(p))
    assert para == {"number_of_random_vectors": 3, "number_of_moments": 1000, "energy_max": 6.1,
                    "calculate_vac": True, "calculate_msd": False}
    p.write_text("calculate_everything\n")
    with pytest.raises(ValueError):
        F.read_para(str(p))
    n = tmp_path / "neighbor.in"
    n.write_text("2 1\n1 1\n2 0 1\n")                                            # count exceeds K_max
    with pytest.raises(ValueError):
        F.read_neighbor(str(n))
    e = tmp_path / "energy.in"
    e.write_text("3\n-1.0\n\n0.0\n1.0\n9.0\n")                                   # count first; extra lines ignored
    assert F.read_column(str(e), counted=True).tolist() == [-1.0, 0.0, 1.0]


def test_out_files_append(tmp_path):
    path = str(tmp_path / "dos.out")
    F.append_rows(path, np.array([0.1, 0.2, 1.0 / 3.0]))
    F.append_rows(path, np.array([[1.0, 2.0, 3.0], [4.0, 5.0, 6.0]]))
    rows = np.loadtxt(path)
    assert rows.shape == (3, 3) and rows[0, 2] == 1.0 / 3.0 and rows[2, 0] == 4.0


class _OracleEngine:
    def __init__(self, oracle_mod, model, batch, modes):
        self.o, self.mod = oracle_mod.Oracle(model, batch=batch, modes=modes), oracle_mod

    def __getattr__(self, name):
        return getattr(self.o, name)

    def running_conductivity(self, kind, corr, dos, dt):
        return self.mod.running_conductivity(kind, corr, dos, dt)

    def localization_length(self, length):
        return self.mod.localization_length(length)


def test_run_folder_and_driver_file(tmp_path, oracle_mod, monkeypatch):
    """run_folder writes one dos row and N_t vac / msd rows per random vector, appends on a second run, and
    the driver file lists several folders."""
    model = L.square(8, 6, W=4.0, seed=3, energy_scale=6.1)
    E = np.linspace(-6.0, 6.0, 13)
    dts = [0.2, 0.2, 0.4]
    folders = [tmp_path / "a", tmp_path / "b"]
    for f in folders:
        F.write_folder(str(f), model, E, dts, {"calculate_vac": True, "calculate_msd": True,
                                               "number_of_random_vectors": 3, "number_of_moments": 40})
    def make(mdl, b, vac, msd):
        modes = (oracle_mod.MODE_VAC if vac else 0) | (oracle_mod.MODE_MSD if msd else 0)
        return _OracleEngine(oracle_mod, mdl, b, modes)
    F.run_folder(str(folders[0]), seed=7, make_engine=make)
    dos, vac, msd = (np.loadtxt(folders[0] / n) for n in ("dos.out", "vac.out", "msd.out"))
    assert dos.shape == (3, 13) and vac.shape == (9, 13) and msd.shape == (9, 13)      # N_r rows; N_r * N_t rows
    # rows of vector 2 (run alone in the second batch of sizes 2 + 1) against direct oracle calls
    phi = F.random_phase_vectors(model.N, 1, 7, first_vector=2)
    o = oracle_mod.Oracle(model, batch=1, modes=oracle_mod.MODE_VAC | oracle_mod.MODE_MSD)
    o.set_state(phi)
    assert np.allclose(dos[2], o.kpm_transform(o.dos_moments(40), E)[0], rtol=0, atol=1e-15)
    assert np.allclose(vac[6], o.kpm_transform(o.vac(40), E)[0], rtol=0, atol=1e-13)    # t = 0 row of vector 2
    F.run_folder(str(folders[0]), seed=7, make_engine=make)                              # append, not overwrite
    assert np.loadtxt(folders[0] / "dos.out").shape == (6, 13)
    # driver input file: folders relative to the file, whitespace separated
    (tmp_path / "input.txt").write_text("a\nb\n")
    calls = []
    monkeypatch.setattr(F, "run_folder", lambda path, **kw: calls.append(os.path.basename(path)))
    assert F.main([str(tmp_path / "input.txt")]) == 0 and calls == ["a", "b"]
