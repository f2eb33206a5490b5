"""File front-end of the paper's program (section 4): the seven `.in` input files of a
simulation folder, the three append-mode `.out` files and the "driver input file" that lists folders.

Host plumbing only (parsing, formatting, call sequencing): every number written to an `.out` file
is produced by libgpuqt.so through `transport.run`.  Site indices in `neighbor.in` are 0-based
("the nth line ... the (n-1)th site", PAPER.md:244 [A11]).

    python -m paper_1705_01387_b200.frontend input.txt          # run every folder listed in input.txt
"""
import os
import sys
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

# para.in defaults
DEFAULTS = {"number_of_random_vectors": 1, "number_of_moments": 1000, "energy_max": 10.0,
            "calculate_vac": False, "calculate_msd": False}


@dataclass
class Model:
    """The four input data sets in the layout gpuqt_create takes."""
    N: int
    K: int
    nbr_count: np.ndarray
    nbr_index: np.ndarray                 # [N*K], unused slots -1
    hop_re: Optional[np.ndarray]
    hop_im: Optional[np.ndarray]
    onsite: Optional[np.ndarray]
    x: np.ndarray
    box_length: float
    volume: float
    energy_scale: float
    name: str = "folder"
    meta: dict = field(default_factory=dict)


def _lines(path):
    with open(path) as f:
        return [ln.split() for ln in f if ln.strip()]


def _fmt(v):
    return repr(float(v))


# ------------------------------------------------------------------------------------------- readers
def read_neighbor(path):
    """neighbor.in: line 1 = N K_max; line n+1 = count, indices of site n-1."""
    rows = _lines(path)
    N, K = int(rows[0][0]), int(rows[0][1])
    if len(rows) - 1 != N:
        raise ValueError(f"{path}: {len(rows) - 1} site lines for N = {N}")
    count = np.zeros(N, np.int32)
    index = np.full((N, K), -1, np.int32)
    for m, r in enumerate(rows[1:]):
        c = int(r[0])
        if c < 0 or c > K or len(r) != c + 1:
            raise ValueError(f"{path}: line {m + 2}: {len(r) - 1} indices for a count of {c} (K_max = {K})")
        count[m] = c
        index[m, :c] = [int(t) for t in r[1:]]
    return N, K, count, index.reshape(-1)


def read_hopping(path, count, K):
    """hopping.in: 'real' or 'complex', then one line per site in neighbour order."""
    with open(path) as f:
        raw = [ln.split() for ln in f]
    while raw and not raw[-1]:
        raw.pop()
    while raw and not raw[0]:
        raw.pop(0)
    kind = raw[0][0].lower() if raw else ""
    if kind not in ("real", "complex"):
        raise ValueError(f"{path}: first line must be 'real' or 'complex'")
    N = count.size
    rows = raw                                    # a site without neighbours has an empty line: keep blank lines
    if len(rows) - 1 != N:
        rows = [raw[0]] + [r for r in raw[1:] if r]            # ... unless the writer dropped them
        it = iter(rows[1:])
        rows = [raw[0]] + [next(it, []) if count[m] > 0 else [] for m in range(N)]
        if next(it, None) is not None:
            raise ValueError(f"{path}: more hopping lines than sites with neighbours")
    re = np.zeros((N, K))
    im = np.zeros((N, K)) if kind == "complex" else None
    per = 2 if kind == "complex" else 1
    for m, r in enumerate(rows[1:]):
        c = int(count[m])
        if len(r) != per * c:
            raise ValueError(f"{path}: line {m + 2}: {len(r)} numbers for {c} neighbours ({kind})")
        vals = [float(t) for t in r]
        re[m, :c] = vals[0::per]
        if im is not None:
            im[m, :c] = vals[1::2]
    return re.reshape(-1), None if im is None else im.reshape(-1)


def read_column(path, counted):
    """potential.in (one value per line) or energy.in / time_step.in (count first, :275-303)."""
    vals = [float(r[0]) for r in _lines(path)]
    if counted:
        n = int(vals[0])
        if len(vals) - 1 < n:
            raise ValueError(f"{path}: {len(vals) - 1} values for a count of {n}")
        return np.array(vals[1:n + 1])
    return np.array(vals)


def read_position(path, N):
    """position.in: line 1 = box length, volume; then X_m per line."""
    rows = _lines(path)
    box, vol = float(rows[0][0]), float(rows[0][1])
    x = np.array([float(r[0]) for r in rows[1:]])
    if x.size != N:
        raise ValueError(f"{path}: {x.size} positions for N = {N}")
    return box, vol, x


def read_para(path):
    """para.in: keyword [value]; blank lines ignored; absent keywords take defaults."""
    p = dict(DEFAULTS)
    if os.path.exists(path):
        for r in _lines(path):
            key = r[0]
            if key in ("calculate_vac", "calculate_msd"):
                p[key] = True
            elif key in ("number_of_random_vectors", "number_of_moments"):
                p[key] = int(r[1])
            elif key == "energy_max":
                p[key] = float(r[1])
            else:
                raise ValueError(f"{path}: unknown keyword '{key}'")
    return p


def read_folder(folder):
    """All input files of one simulation folder -> (Model, para dict, energies, time steps or None)."""
    j = lambda name: os.path.join(folder, name)
    para = read_para(j("para.in"))
    N, K, count, index = read_neighbor(j("neighbor.in"))
    hop_re = hop_im = onsite = None
    if os.path.exists(j("hopping.in")):                       # optional: all hoppings -1
        hop_re, hop_im = read_hopping(j("hopping.in"), count, K)
    if os.path.exists(j("potential.in")):                     # optional: all on-site potentials 0
        onsite = read_column(j("potential.in"), counted=False)
        if onsite.size != N:
            raise ValueError(f"potential.in: {onsite.size} values for N = {N}")
    box, vol, x = read_position(j("position.in"), N)
    energies = read_column(j("energy.in"), counted=True)
    dts = None
    if para["calculate_vac"] or para["calculate_msd"]:        # otherwise time_step.in is not needed
        dts = read_column(j("time_step.in"), counted=True)
    model = Model(N=N, K=K, nbr_count=count, nbr_index=index, hop_re=hop_re, hop_im=hop_im, onsite=onsite, x=x,
                  box_length=box, volume=vol, energy_scale=para["energy_max"], name=os.path.basename(folder.rstrip("/")))
    return model, para, energies, dts


# ------------------------------------------------------------------------------------------- writers
def write_folder(folder, model, energies, dts=None, para=None):
    """Write a simulation folder in the paper's formats (what its make_inputs.cpp programs produce)."""
    os.makedirs(folder, exist_ok=True)
    j = lambda name: os.path.join(folder, name)
    N, K = model.N, model.K
    idx = np.asarray(model.nbr_index).reshape(N, K)
    with open(j("neighbor.in"), "w") as f:
        f.write(f"{N} {K}\n")
        for m in range(N):
            c = int(model.nbr_count[m])
            f.write(" ".join([str(c)] + [str(int(t)) for t in idx[m, :c]]) + "\n")
    if model.hop_re is not None:
        re = np.asarray(model.hop_re).reshape(N, K)
        im = None if model.hop_im is None else np.asarray(model.hop_im).reshape(N, K)
        with open(j("hopping.in"), "w") as f:
            f.write("real\n" if im is None else "complex\n")
            for m in range(N):
                c = int(model.nbr_count[m])
                if im is None:
                    f.write(" ".join(_fmt(v) for v in re[m, :c]) + "\n")
                else:
                    f.write(" ".join(f"{_fmt(a)} {_fmt(b)}" for a, b in zip(re[m, :c], im[m, :c])) + "\n")
    if model.onsite is not None:
        with open(j("potential.in"), "w") as f:
            f.writelines(_fmt(v) + "\n" for v in model.onsite)
    with open(j("position.in"), "w") as f:
        f.write(f"{_fmt(model.box_length)} {_fmt(model.volume)}\n")
        f.writelines(_fmt(v) + "\n" for v in model.x)
    with open(j("energy.in"), "w") as f:
        f.write(f"{len(energies)}\n")
        f.writelines(_fmt(v) + "\n" for v in energies)
    if dts is not None:
        with open(j("time_step.in"), "w") as f:
            f.write(f"{len(dts)}\n")
            f.writelines(_fmt(v) + "\n" for v in dts)
    para = dict(para or {})
    para.setdefault("energy_max", model.energy_scale)
    with open(j("para.in"), "w") as f:
        for key, val in para.items():
            if key in ("calculate_vac", "calculate_msd"):
                if val:
                    f.write(key + "\n\n")
            else:
                f.write(f"{key} {val!r}\n")


def append_rows(path, rows):
    """dos.out / vac.out / msd.out: one row per line, column n = energy point n; APPEND."""
    with open(path, "a") as f:
        for row in np.atleast_2d(rows):
            f.write(" ".join(_fmt(v) for v in row) + "\n")


# ------------------------------------------------------------------------------------------- driver
def random_phase_vectors(N, count, seed, first_vector=0):
    """phi_i = exp(i theta_i), theta uniform (PAPER.md:140 [A7]); one generator stream per vector."""
    out = np.empty((count, N, 2))
    for b in range(count):
        theta = np.random.default_rng([seed, first_vector + b]).uniform(0.0, 2.0 * np.pi, N)
        out[b, :, 0], out[b, :, 1] = np.cos(theta), np.sin(theta)
    return out


def run_folder(folder, seed=170501387, make_engine=None, batch=None):
    """Run one simulation folder: N_r random vectors in batches of B, results appended to dos.out, vac.out
    (N_t rows per vector, rho C_vv at t_k) and msd.out (N_t rows per vector, rho dX^2 at t_{k+1}).
    `make_engine(model, batch, vac, msd)` defaults to the CUDA library."""
    from . import binding, transport
    model, para, energies, dts = read_folder(folder)
    vac, msd = para["calculate_vac"], para["calculate_msd"]
    n_r, nm = para["number_of_random_vectors"], para["number_of_moments"]
    B = batch or max(b for b in (8, 4, 2, 1) if b <= n_r)
    if make_engine is None:
        def make_engine(mdl, b, want_vac, want_msd):
            modes = (binding.MODE_VAC if want_vac else 0) | (binding.MODE_MSD if want_msd else 0)
            return binding.GpuQT(mdl, batch=b, modes=modes)
    order_of = lambda dt: binding.choose_order(model.energy_scale, dt)
    done = 0
    while done < n_r:
        b = max(x for x in (8, 4, 2, 1) if x <= min(B, n_r - done))
        eng = make_engine(model, b, vac, msd)
        phi = random_phase_vectors(model.N, b, seed, done)
        res = transport.run(eng, phi, dts if dts is not None else [], nm, energies, order_of, vac=vac, msd=msd,
                            per_vector=True)
        for v in range(b):                                     # one block of rows per random vector
            append_rows(os.path.join(folder, "dos.out"), res["dos"][v])
            if vac:
                append_rows(os.path.join(folder, "vac.out"), res["rho_vac"][:, v, :])
            if msd:
                append_rows(os.path.join(folder, "msd.out"), res["rho_msd"][:, v, :])
        if hasattr(eng, "close"):
            eng.close()
        done += b
    return para


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    if len(argv) != 1:
        print("usage: python -m paper_1705_01387_b200.frontend <driver input file>", file=sys.stderr)
        return 2
    base = os.path.dirname(os.path.abspath(argv[0]))
    with open(argv[0]) as f:
        folders = [tok for ln in f for tok in ln.split()]
    for folder in folders:                                     # "run the two examples consecutively"
        path = folder if os.path.isabs(folder) else os.path.join(base, folder)
        if not os.path.isdir(path):
            path = folder                                      # relative to the working directory, as the paper's command
        print(f"gpuqt: running {path}", flush=True)
        run_folder(path)
    return 0


if __name__ == "__main__":
    sys.exit(main())
