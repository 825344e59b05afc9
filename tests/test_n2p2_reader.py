"""n2p2 model reader (paper_2002_00054_b200/n2p2.py, PAPER.md L54 / L58): the tests WRITE
their own input.nn / scaling.data / weights.NNN.data fixtures from a workloads.Model (no n2p2 model file exists in
this container -- the format readings R1-R5 in that module are unverified against a real one) and check that
reading them back gives the same nnp_create arguments, and that the oracle evaluates both to the same numbers.
CPU only; the GPU side of the same round trip is tests/test_gpu_parity.py::test_n2p2_model_round_trip."""
import os

import numpy as np
import pytest

import oracle
import workloads as W
from paper_2002_00054_b200 import n2p2

Z = {"H": 1, "O": 8, "Ni": 28}


def write_model(directory, model, order=None, indexed=True, scaling_mode=None, smin=0.0, smax=1.0,
                atom_energy=None, conv=None, extra=(), sorted_inputs=True):
    """Fixture writer (tests only).  `order`: permutation applied to the symfunction_short lines per element (any
    order may appear in input.nn).  sorted_inputs=True: the weight and scaling files refer to the network inputs in
    n2p2's SORTED symmetry-function order (reading R2), as n2p2 writes them; False: in the order of the lines.
    `scaling_mode`: None | "scale" | "center" | "scalecenter" | "sigma"."""
    os.makedirs(directory, exist_ok=True)
    lines_model = model
    if sorted_inputs:
        model = _sorted_model(model)
    names = list(model.elements)
    conv_e, conv_l, mean_e = conv if conv else (1.0, 1.0, 0.0)
    act = {"softplus": "p", "tanh": "t"}[model.activation]
    nodes = model.layer_sizes[0][1:-1]
    with open(os.path.join(directory, "input.nn"), "w") as fh:
        fh.write("# fixture written by tests/test_n2p2_reader.py\n")
        fh.write("number_of_elements %d\n" % len(names))
        fh.write("elements %s   # any order in the file\n" % " ".join(reversed(names)))
        for nm, e in (atom_energy or {}).items():
            fh.write("atom_energy %s %.17g\n" % (nm, e))
        fh.write("cutoff_type 1\nrandom_seed 1234\nepochs 10\n")
        if conv:
            fh.write("mean_energy %.17g\nconv_energy %.17g\nconv_length %.17g\n" % (mean_e, conv_e, conv_l))
        fh.write("global_hidden_layers_short %d\n" % len(nodes))
        fh.write("global_nodes_short %s\n" % " ".join(str(x) for x in nodes))
        fh.write("global_activation_short %s l\n" % " ".join([act] * len(nodes)))
        if scaling_mode in ("scale", "scalecenter"):
            fh.write("scale_symmetry_functions\n")
        if scaling_mode in ("center", "scalecenter"):
            fh.write("center_symmetry_functions\n")
        if scaling_mode == "sigma":
            fh.write("scale_symmetry_functions_sigma\n")
        if scaling_mode:
            fh.write("scale_min_short %.17g\nscale_max_short %.17g\n" % (smin, smax))
        for line in extra:
            fh.write(line + "\n")
        lm = lines_model
        rcs = lm.sf_cutoffs if lm.sf_cutoffs is not None else [lm.rc] * len(lm.sf)
        for c in range(len(names)):
            idx = [q for q in range(len(lm.sf)) if lm.sf["central"][q] == c]
            if order is not None:
                idx = [idx[k] for k in order(len(idx))]
            for q in idx:
                f = lm.sf[q]
                eta, rs, rc = f["eta"] / conv_l ** 2, f["rs"] * conv_l, rcs[q] * conv_l      # file units
                if f["kind"] == 2:
                    fh.write("symfunction_short %s 2 %s %.17g %.17g %.17g\n" % (names[c], names[f["e1"]], eta, rs, rc))
                else:
                    fh.write("symfunction_short %s %d %s %s %.17g %.17g %.17g %.17g\n"
                             % (names[c], f["kind"], names[f["e2"]], names[f["e1"]], eta, f["lam"], f["zeta"], rc))
    for c, nm in enumerate(names):
        sizes = model.layer_sizes[c]
        w = np.array(model.weights[c], dtype=np.float64).copy()
        n_last = sizes[-2]
        # the files hold the network in n2p2's normalised units; mean_energy and atom_energy come ON TOP (reading R5)
        w[-1] *= conv_e
        w[-(n_last + 1):-1] *= conv_e
        with open(os.path.join(directory, "weights.%03d.data" % Z[nm]), "w") as fh:
            fh.write("# value type index l_s n_s l_e n_e\n")
            pos, k = 0, 0
            for l in range(len(sizes) - 1):
                Wl = w[pos:pos + sizes[l] * sizes[l + 1]].reshape(sizes[l + 1], sizes[l]); pos += Wl.size
                bl = w[pos:pos + sizes[l + 1]]; pos += bl.size
                for i in range(sizes[l]):
                    for j in range(sizes[l + 1]):
                        k += 1
                        fh.write("%24.16E a %9d %4d %4d %4d %4d\n" % (Wl[j, i], k, l, i + 1, l + 1, j + 1) if indexed
                                 else "%24.16E\n" % Wl[j, i])
                for j in range(sizes[l + 1]):
                    k += 1
                    fh.write("%24.16E b %9d %4d %4d\n" % (bl[j], k, l + 1, j + 1) if indexed else "%24.16E\n" % bl[j])
    if scaling_mode:
        with open(os.path.join(directory, "scaling.data"), "w") as fh:
            fh.write("# e_index sf_index min max mean sigma\n")
            for c in range(len(names)):
                shift, scale = model.sf_scaling[c]
                for s in range(len(shift)):
                    # choose statistics that reproduce x = scale (G - shift) under the mode's formula (reading R4)
                    if scaling_mode == "scale":          # x = smin + (smax-smin)(G-gmin)/(gmax-gmin)
                        rng_ = (smax - smin) / scale[s]; gmin = shift[s] + smin / scale[s]; row = (gmin, gmin + rng_, 0.123, 0.456)
                    elif scaling_mode == "center":       # x = G - gmean
                        row = (-1.0, 2.0, shift[s], 0.5)
                    elif scaling_mode == "scalecenter":  # x = smin + (smax-smin)(G-gmean)/(gmax-gmin)
                        rng_ = (smax - smin) / scale[s]; row = (0.25, 0.25 + rng_, shift[s] + smin / scale[s], 0.7)
                    else:                                # sigma: x = smin + (smax-smin)(G-gmean)/sigma
                        row = (0.0, 1.0, shift[s] + smin / scale[s], (smax - smin) / scale[s])
                    fh.write("%10d %10d %24.16E %24.16E %24.16E %24.16E\n" % ((c + 1, s + 1) + row))
            fh.write("%24.16E %24.16E\n" % (-1.5, 0.3))   # energy statistics line: ignored


def _sorted_model(model):
    """The same model with every element's symmetry functions in the reader's sort order (reading R2) and the first
    network layer / scaling permuted accordingly -- what read_model(sort='n2p2') must return."""
    import copy
    m = copy.deepcopy(model)
    rcs = np.array(model.sf_cutoffs if model.sf_cutoffs is not None else [model.rc] * len(model.sf))
    new_sf, new_rc = [], []
    for c in range(len(model.elements)):
        idx = [q for q in range(len(model.sf)) if model.sf["central"][q] == c]
        key = lambda q: (model.sf["kind"][q], rcs[q], model.sf["eta"][q], model.sf["rs"][q], model.sf["zeta"][q],
                         model.sf["lam"][q], model.sf["e1"][q], model.sf["e2"][q])
        perm = sorted(range(len(idx)), key=lambda k: key(idx[k]))
        new_sf += [model.sf[idx[k]] for k in perm]
        new_rc += [rcs[idx[k]] for k in perm]
        sizes = model.layer_sizes[c]
        w = np.array(model.weights[c]).copy()
        W1 = w[:sizes[0] * sizes[1]].reshape(sizes[1], sizes[0])[:, perm]
        w[:sizes[0] * sizes[1]] = W1.ravel()
        m.weights[c] = w
        if model.sf_scaling is not None:
            m.sf_scaling[c] = (np.asarray(model.sf_scaling[c][0])[perm], np.asarray(model.sf_scaling[c][1])[perm])
    m.sf = np.array(new_sf, dtype=model.sf.dtype)
    m.sf_cutoffs = None if model.sf_cutoffs is None else list(new_rc)
    return m


def _assert_same(a, b, tol=0.0):
    assert tuple(a.elements) == tuple(b.elements)
    assert a.rc == pytest.approx(b.rc, rel=1e-15)
    for k in ("central", "kind", "e1", "e2"):
        assert np.array_equal(a.sf[k], b.sf[k]), k
    for k in ("eta", "rs", "lam", "zeta"):
        assert np.allclose(a.sf[k], b.sf[k], rtol=max(tol, 4e-16), atol=0.0), k
    assert [list(x) for x in a.layer_sizes] == [list(x) for x in b.layer_sizes]
    for wa, wb in zip(a.weights, b.weights):
        assert np.allclose(wa, wb, rtol=max(tol, 1e-15), atol=1e-300)
    assert a.activation == b.activation
    assert (a.sf_cutoffs is None) == (b.sf_cutoffs is None)
    if a.sf_cutoffs is not None:
        assert np.allclose(a.sf_cutoffs, b.sf_cutoffs, rtol=4e-16)
    assert (a.sf_scaling is None) == (b.sf_scaling is None)
    if a.sf_scaling is not None:
        for (s1, c1), (s2, c2) in zip(a.sf_scaling, b.sf_scaling):
            assert np.allclose(s1, s2, rtol=1e-12, atol=1e-13) and np.allclose(c1, c2, rtol=1e-12)


@pytest.mark.parametrize("indexed", [True, False])
def test_round_trip_base_model(tmp_path, indexed):
    model = W.make_model(False)
    write_model(str(tmp_path), model, order=lambda n: list(np.random.RandomState(1).permutation(n)), indexed=indexed)
    got = n2p2.read_model(str(tmp_path))
    _assert_same(got, _sorted_model(model))
    assert got.atomic_numbers == (1, 8) and got.n_sf_per_elem == [52, 52]
    # the kernels the read model would run on: still the specialised base-12 shape
    from paper_2002_00054_b200.binding import table_kernels
    assert table_kernels(got) == ("base12", "base12")
    # file order instead of n2p2's sort
    write_model(str(tmp_path), model, indexed=indexed, sorted_inputs=False)
    _assert_same(n2p2.read_model(str(tmp_path), sort="file"), model)


@pytest.mark.parametrize("mode", ["scale", "center", "scalecenter", "sigma"])
def test_scaling_modes_fold_into_affine_form(tmp_path, mode):
    import copy
    model = copy.deepcopy(W.make_model(False, elements=("H", "O"), hidden=(6, 5)))
    rs = np.random.RandomState(3)
    if mode == "center":
        model.sf_scaling = [(rs.uniform(0.0, 0.5, n), np.ones(n)) for n in model.n_sf_per_elem]
    else:
        model.sf_scaling = [(rs.uniform(0.0, 0.5, n), rs.uniform(0.2, 3.0, n)) for n in model.n_sf_per_elem]
    model.activation = "tanh"
    smin, smax = (0.0, 1.0) if mode == "center" else (-0.5, 1.5)
    if mode == "center":
        smin = 0.0
    write_model(str(tmp_path), model, scaling_mode=mode, smin=smin, smax=smax)
    got = n2p2.read_model(str(tmp_path))
    _assert_same(got, _sorted_model(model))


def test_oracle_energy_and_forces_survive_the_round_trip(tmp_path):
    # per-SF cutoff radii, wide angular SFs, atom_energy offsets and normalisation (conv_energy / conv_length /
    # mean_energy) all folded by the reader: the ORACLE must give the same E and F on the original model
    # (+ offsets) and on the one read back from the files
    from conftest import tiny_model
    rows, rcs = [], []
    for c in range(2):
        for e1 in range(2):
            for rr, eta in ((6.0, 0.03), (4.5, 0.2)):
                rows.append((c, 2, e1, 0, eta, 0.4, 0.0, 0.0)); rcs.append(rr)
        for (e1, e2) in ((0, 0), (0, 1), (1, 1)):
            rows.append((c, 3, e1, e2, 0.01, 0.0, 1.0, 2.0)); rcs.append(6.0)
            rows.append((c, 3, e1, e2, 0.002, 0.0, -1.0, 4.0)); rcs.append(5.0)
            rows.append((c, 9, e1, e2, 0.02, 0.0, 1.0, 1.0)); rcs.append(4.0)
    model = tiny_model(rows, n_elem=2, hidden=(5, 4), seed=31)
    model.elements = ("H", "O")
    model.sf_cutoffs = rcs
    offs = {"H": -0.4581, "O": -2.0413}
    write_model(str(tmp_path), model, atom_energy=offs, conv=(27.2114, 1.8897261, -0.125),
                order=lambda n: list(range(n))[::-1])
    got = n2p2.read_model(str(tmp_path))
    assert not np.array_equal(got.sf, model.sf)          # the reader did re-order the table ...
    sysm = W.make_water(40, 5, L=12.6)
    ref = oracle.compute(oracle.OracleModel(model), sysm.pos, sysm.types, sysm.box)      # ... and the physics is the same
    res = oracle.compute(oracle.OracleModel(got), sysm.pos, sysm.types, sysm.box)
    e_off = sum(offs[model.elements[t]] for t in sysm.types) + (-0.125) * sysm.n_atoms      # atom_energy + mean_energy
    assert res.e_total == pytest.approx(ref.e_total + e_off, rel=1e-12)
    assert np.abs(res.F - ref.F).max() <= 1e-11 * max(1.0, np.abs(ref.F).max())
    assert np.abs(ref.F).max() > 1e-4


def test_rejects_what_it_cannot_represent(tmp_path):
    model = W.make_model(False, hidden=(4, 3))
    d = str(tmp_path)
    write_model(d, model, extra=["cutoff_type 2 0.5"])             # later line wins: tanh cutoff
    with pytest.raises(n2p2.N2P2Error, match="cutoff_type"):
        n2p2.read_model(d)
    write_model(d, model, extra=["symfunction_short H 12 0.01 0.0 6.0"])
    with pytest.raises(n2p2.N2P2Error, match="type 12"):
        n2p2.read_model(d)
    write_model(d, model, extra=["normalize_nodes"])
    with pytest.raises(n2p2.N2P2Error, match="normalize_nodes"):
        n2p2.read_model(d)
    write_model(d, model)
    os.remove(os.path.join(d, "weights.008.data"))
    with pytest.raises(n2p2.N2P2Error, match="weights.008.data"):
        n2p2.read_model(d)
    write_model(d, model)
    with open(os.path.join(d, "weights.001.data"), "a") as fh:
        fh.write("0.5 a 999 0 1 1 1\n")
    with pytest.raises(n2p2.N2P2Error, match="values"):
        n2p2.read_model(d)
    model.sf_scaling = [(np.zeros(n), np.ones(n)) for n in model.n_sf_per_elem]
    write_model(d, model, scaling_mode="scale")                    # scaling requested, file incomplete
    lines = open(os.path.join(d, "scaling.data")).read().splitlines()
    open(os.path.join(d, "scaling.data"), "w").write("\n".join(lines[:-5]) + "\n")
    with pytest.raises(n2p2.N2P2Error, match="incomplete"):
        n2p2.read_model(d)
