"""Reader for n2p2 model directories (input.nn, scaling.data, weights.NNN.data) -> the arguments of nnp_create.

PAPER.md L54: CabanaMD-NNP "re-implement[s] ... from the n2p2 package", L58: and keeps n2p2 for "initialization and
other functionality that is not performance critical" (parsing the model files).  This module is that host-side
initialisation: pure text parsing and re-arrangement of numbers into the `nnp_sf` table, the row-major weight
blocks and the affine symmetry-function scaling of include/nnp.h.  None of the method's arithmetic lives here (no
symmetry function, network or force is evaluated) and nothing here runs per time step.

    model = read_model("path/to/model_dir")        # a workloads.Model-like object
    nnp = NNP.from_model(model)

What is read (n2p2's documented keywords; every other keyword that changes the potential raises N2P2Error, purely
informational / training keywords are ignored):
  number_of_elements, elements, atom_energy, cutoff_type (1 = cosine, alpha 0 only), symfunction_short of type 2
  (radial), 3 (angular narrow), 9 (angular wide), global_hidden_layers_short, global_nodes_short,
  global_activation_short (hidden: all "t" = tanh or all "p" = softplus; output "l"), scale_symmetry_functions,
  scale_symmetry_functions_sigma, center_symmetry_functions, scale_min_short, scale_max_short, mean_energy,
  conv_energy, conv_length.

Readings ("n2p2 files"; UNVERIFIED AGAINST A REAL MODEL -- no n2p2 model file exists in this
container, the tests write their own fixtures):
  R1  elements are ordered by atomic number; element index = position in that order.
  R2  the symmetry functions of an element are SORTED before they meet the network inputs and the rows of
      scaling.data, by the key (type, rc, eta, rs, [zeta, lambda,] e1 [, e2]) ascending (n2p2 sorts its
      SymFnc objects; the published key order is type, cutoff, eta, rs, then the angular parameters, then the
      neighbour elements).  `sort="file"` keeps the order of input.nn instead.
  R3  weights.NNN.data lists, layer by layer, the weights a(i -> j) with the SOURCE neuron i as the outer loop,
      then the biases b(j) of the layer.  When a line carries n2p2's index columns
      (value, "a", index, l_s, n_s, l_e, n_e  /  value, "b", index, l, n) those are used instead of the position.
  R4  scaling.data rows: element index (1-based), SF index (1-based, sorted order), min, max, mean, sigma.
      scale only:        x = Smin + (Smax - Smin) (G - Gmin) / (Gmax - Gmin)
      center only:       x = G - Gmean
      scale + center:    x = Smin + (Smax - Smin) (G - Gmean) / (Gmax - Gmin)
      scale with sigma:  x = Smin + (Smax - Smin) (G - Gmean) / sigma
      all folded into x = scale (G - shift) of nnp_set_sf_scaling.
  R5  atom_energy offsets and the normalisation keywords are folded into the model: with conv_length L and
      conv_energy C (file units = physical units x conv), eta_phys = eta L^2, rs_phys = rs / L, rc_phys = rc / L,
      output layer (w, b) -> (w / C, b / C + mean_energy + atom_energy).
"""
from __future__ import annotations

import os
from dataclasses import dataclass, field

import numpy as np

SF_DTYPE = np.dtype(
    [("central", "<i4"), ("kind", "<i4"), ("e1", "<i4"), ("e2", "<i4"),
     ("eta", "<f8"), ("rs", "<f8"), ("lam", "<f8"), ("zeta", "<f8")],
    align=True,
)

ATOMIC_NUMBER = {s: z + 1 for z, s in enumerate(
    "H He Li Be B C N O F Ne Na Mg Al Si P S Cl Ar K Ca Sc Ti V Cr Mn Fe Co Ni Cu Zn Ga Ge As Se Br Kr Rb Sr Y Zr Nb Mo "
    "Tc Ru Rh Pd Ag Cd In Sn Sb Te I Xe Cs Ba La Ce Pr Nd Pm Sm Eu Gd Tb Dy Ho Er Tm Yb Lu Hf Ta W Re Os Ir Pt Au Hg Tl "
    "Pb Bi Po At Rn".split())}

IGNORED = {  # training / bookkeeping keywords that do not change the potential
    "random_seed", "epochs", "updater_type", "parallel_mode", "jacobian_mode", "update_strategy", "selection_mode",
    "task_batch_size_energy", "task_batch_size_force", "memorize_symfunc_results", "test_fraction",
    "force_weight", "short_energy_fraction", "short_force_fraction", "short_energy_error_threshold",
    "short_force_error_threshold", "rmse_threshold_trials", "use_short_forces", "weights_min", "weights_max",
    "precondition_weights", "nguyen_widrow_weights_short", "write_trainpoints", "write_trainforces",
    "write_weights_epoch", "write_neuronstats", "write_trainlog", "kalman_type", "kalman_epsilon", "kalman_q0",
    "kalman_qtau", "kalman_qmin", "kalman_eta", "kalman_etatau", "kalman_etamax", "kalman_lambda_short",
    "kalman_nue_short", "gradient_type", "gradient_eta", "gradient_adam_eta", "gradient_adam_beta1",
    "gradient_adam_beta2", "gradient_adam_epsilon", "use_old_weights_short", "main_error_metric",
    "rmse_threshold", "rmse_threshold_energy", "rmse_threshold_force", "normalize_data_set",
}


class N2P2Error(ValueError):
    pass


@dataclass
class N2P2Model:
    """Same attributes as workloads.Model (what NNP.from_model and the tests read)."""
    elements: tuple
    rc: float
    sf: np.ndarray
    layer_sizes: list
    weights: list
    name: str = "n2p2"
    n_sf_per_elem: list = field(default_factory=list)
    sf_scaling: list | None = None
    activation: str = "softplus"
    sf_cutoffs: list | None = None
    atomic_numbers: tuple = ()


def _lines(path):
    with open(path) as fh:
        for raw in fh:
            line = raw.split("#", 1)[0].strip()
            if line:
                yield line.split()


def parse_input_nn(path):
    """-> dict of the settings this library needs (strings as in the file)."""
    st = {"symfunction_short": [], "atom_energy": {}, "flags": set()}
    for t in _lines(path):
        key, args = t[0], t[1:]
        if key == "symfunction_short":
            st["symfunction_short"].append(args)
        elif key == "atom_energy":
            st["atom_energy"][args[0]] = float(args[1])
        elif key in ("scale_symmetry_functions", "scale_symmetry_functions_sigma", "center_symmetry_functions"):
            st["flags"].add(key)
        elif key in ("number_of_elements", "elements", "cutoff_type", "global_hidden_layers_short", "global_nodes_short",
                     "global_activation_short", "scale_min_short", "scale_max_short", "mean_energy", "conv_energy",
                     "conv_length"):
            st[key] = args
        elif key in IGNORED:
            continue
        elif key in ("normalize_nodes", "element_nodes_short", "element_hidden_layers_short", "element_activation_short",
                     "symfunction_long", "use_electrostatics", "ewald_type", "nnp_type", "global_hidden_layers_long"):
            raise N2P2Error("input.nn keyword '%s' is not supported by this library" % key)
        # anything else: unknown to this reader; n2p2 has many logging keywords -> ignore
    for need in ("number_of_elements", "elements", "global_hidden_layers_short", "global_nodes_short",
                 "global_activation_short"):
        if need not in st:
            raise N2P2Error("input.nn: missing keyword '%s'" % need)
    return st


def _sf_key(row):
    # reading R2: (type, rc, eta, rs, [zeta, lambda,] e1, e2)
    kind, e1, e2, eta, rs, lam, zeta, rc = row
    return (kind, rc, eta, rs, zeta, lam, e1, e2)


def read_model(directory, sort="n2p2"):
    st = parse_input_nn(os.path.join(directory, "input.nn"))
    n_elem = int(st["number_of_elements"][0])
    names = list(st["elements"])
    if len(names) != n_elem:
        raise N2P2Error("elements: expected %d names" % n_elem)
    for nm in names:
        if nm not in ATOMIC_NUMBER:
            raise N2P2Error("unknown element '%s'" % nm)
    names.sort(key=lambda s: ATOMIC_NUMBER[s])                      # reading R1
    eidx = {s: k for k, s in enumerate(names)}
    ct = st.get("cutoff_type", ["1"])
    if int(ct[0]) != 1 or (len(ct) > 1 and float(ct[1]) != 0.0):
        raise N2P2Error("only cutoff_type 1 (cosine) with alpha = 0 is supported, got %s" % " ".join(ct))
    conv_l = float(st.get("conv_length", ["1.0"])[0])
    conv_e = float(st.get("conv_energy", ["1.0"])[0])
    mean_e = float(st.get("mean_energy", ["0.0"])[0])

    per = [[] for _ in range(n_elem)]          # rows (kind, e1, e2, eta, rs, lam, zeta, rc) in file units
    for a in st["symfunction_short"]:
        try:
            c, kind = eidx[a[0]], int(a[1])
            if kind == 2:
                e1, eta, rs, rc = eidx[a[2]], float(a[3]), float(a[4]), float(a[5])
                per[c].append((2, e1, 0, eta, rs, 0.0, 0.0, rc))
            elif kind in (3, 9):
                e1, e2 = sorted((eidx[a[2]], eidx[a[3]]))
                eta, lam, zeta, rc = float(a[4]), float(a[5]), float(a[6]), float(a[7])
                rs = float(a[8]) if len(a) > 8 else 0.0
                if rs != 0.0:
                    raise N2P2Error("angular symmetry functions with a shift r_s are not supported")
                per[c].append((kind, e1, e2, eta, 0.0, lam, zeta, rc))
            else:
                raise N2P2Error("symfunction_short type %d is not supported (2, 3, 9 are)" % kind)
        except (KeyError, IndexError) as ex:
            raise N2P2Error("bad symfunction_short line: %s" % " ".join(a)) from ex
    for c in range(n_elem):
        if not per[c]:
            raise N2P2Error("element %s has no symmetry functions" % names[c])
        if sort == "n2p2":
            per[c].sort(key=_sf_key)
        elif sort != "file":
            raise ValueError("sort must be 'n2p2' or 'file'")

    rows, rcs = [], []
    for c in range(n_elem):
        for (kind, e1, e2, eta, rs, lam, zeta, rc) in per[c]:
            rows.append((c, kind, e1, e2, eta * conv_l * conv_l, rs / conv_l, lam, zeta))   # reading R5
            rcs.append(rc / conv_l)
    sf = np.array(rows, dtype=SF_DTYPE)
    rc_max = max(rcs)
    n_per = [len(per[c]) for c in range(n_elem)]

    # ---- networks
    n_hidden = int(st["global_hidden_layers_short"][0])
    nodes = [int(x) for x in st["global_nodes_short"]]
    acts = list(st["global_activation_short"])
    if len(nodes) != n_hidden or len(acts) != n_hidden + 1:
        raise N2P2Error("global_nodes_short / global_activation_short do not match global_hidden_layers_short")
    if acts[-1] != "l" or len(set(acts[:-1])) > 1 or (acts[:-1] and acts[0] not in ("t", "p")):
        raise N2P2Error("activations must be all 't' (tanh) or all 'p' (softplus) on the hidden layers and 'l' on the output")
    activation = "tanh" if acts[:-1] and acts[0] == "t" else "softplus"
    layer_sizes, weights = [], []
    for c in range(n_elem):
        sizes = [n_per[c], *nodes, 1]
        path = os.path.join(directory, "weights.%03d.data" % ATOMIC_NUMBER[names[c]])
        w = _read_weights(path, sizes)
        off = mean_e + st["atom_energy"].get(names[c], 0.0)
        # output layer: (w, b) -> (w / conv_energy, b / conv_energy + mean_energy + atom_energy)     (reading R5)
        n_last = sizes[-2]
        w[-(n_last + 1):-1] /= conv_e
        w[-1] = w[-1] / conv_e + off
        layer_sizes.append(sizes)
        weights.append(w)

    # ---- scaling
    scaling = None
    flags = st["flags"]
    if flags:
        smin = float(st.get("scale_min_short", ["0.0"])[0])
        smax = float(st.get("scale_max_short", ["1.0"])[0])
        table = _read_scaling(os.path.join(directory, "scaling.data"), n_per)
        scaling = []
        for c in range(n_elem):
            gmin, gmax, gmean, gsig = (table[c][:, k] for k in range(4))
            if "scale_symmetry_functions_sigma" in flags:
                scale, centre, lo = (smax - smin) / gsig, gmean, smin
            elif "scale_symmetry_functions" in flags:
                scale = (smax - smin) / (gmax - gmin)
                centre, lo = (gmean, smin) if "center_symmetry_functions" in flags else (gmin, smin)
            else:                                   # center only
                scale, centre, lo = np.ones_like(gmean), gmean, 0.0
            if not np.all(np.isfinite(scale)) or np.any(scale == 0.0):
                raise N2P2Error("scaling.data: a symmetry function has zero range / sigma")
            scaling.append((centre - lo / scale, scale))          # x = scale (G - centre) + lo
    return N2P2Model(elements=tuple(names), rc=rc_max, sf=sf, layer_sizes=layer_sizes, weights=weights,
                     name="n2p2:" + os.path.basename(os.path.normpath(directory)), n_sf_per_elem=n_per,
                     sf_scaling=scaling, activation=activation,
                     sf_cutoffs=None if all(r == rc_max for r in rcs) else rcs,
                     atomic_numbers=tuple(ATOMIC_NUMBER[s] for s in names))


def _read_weights(path, sizes):
    """-> flat row-major [W1[out][in], b1, W2, b2, ...] (include/nnp.h).  Reading R3."""
    if not os.path.exists(path):
        raise N2P2Error("missing weight file %s" % path)
    entries = list(_lines(path))
    n_expected = sum(a * b + b for a, b in zip(sizes[:-1], sizes[1:]))
    if len(entries) != n_expected:
        raise N2P2Error("%s: %d values, the architecture %s needs %d" % (path, len(entries), sizes, n_expected))
    W = [np.full((sizes[l + 1], sizes[l]), np.nan) for l in range(len(sizes) - 1)]
    B = [np.full(sizes[l + 1], np.nan) for l in range(len(sizes) - 1)]
    indexed = all(len(t) >= 5 and t[1] in ("a", "b") for t in entries)
    if indexed:
        for t in entries:
            v = float(t[0])
            if t[1] == "a":
                ls, ns, le, ne = int(t[3]), int(t[4]), int(t[5]), int(t[6])
                if le != ls + 1:
                    raise N2P2Error("%s: weight between non-adjacent layers" % path)
                W[ls][ne - 1, ns - 1] = v
            else:
                l, nn = int(t[3]), int(t[4])
                B[l - 1][nn - 1] = v
    else:
        pos = 0
        for l in range(len(sizes) - 1):
            for i in range(sizes[l]):                  # source neuron: outer loop
                for j in range(sizes[l + 1]):
                    W[l][j, i] = float(entries[pos][0]); pos += 1
            for j in range(sizes[l + 1]):
                B[l][j] = float(entries[pos][0]); pos += 1
    flat = np.concatenate([np.concatenate([W[l].ravel(), B[l]]) for l in range(len(sizes) - 1)])
    if not np.all(np.isfinite(flat)):
        raise N2P2Error("%s: missing or non-finite weights" % path)
    return flat


def _read_scaling(path, n_per):
    if not os.path.exists(path):
        raise N2P2Error("scaling requested in input.nn but %s is missing" % path)
    table = [np.full((n, 4), np.nan) for n in n_per]
    for t in _lines(path):
        if len(t) != 6:
            continue                                   # trailing energy statistics line(s)
        e, s = int(t[0]) - 1, int(t[1]) - 1
        if not (0 <= e < len(n_per) and 0 <= s < n_per[e]):
            raise N2P2Error("scaling.data: index (%d, %d) out of range" % (e + 1, s + 1))
        table[e][s] = [float(x) for x in t[2:6]]
    for e, tb in enumerate(table):
        if not np.all(np.isfinite(tb)):
            raise N2P2Error("scaling.data: element %d is incomplete" % (e + 1))
    return table
