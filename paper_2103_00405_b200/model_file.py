"""Front end for the paper's model-file format (Table 4, :274-288; described at :187).

    // comment
    # init
    A = 1000
    B = 1000
    # reactions
    1 A - -> 2 A : 10
    1 A 1 B - -> 2 B : 0.01
    1 B - -> NULL : 10
    # end
    time = 2
    steps = 10000

Each reaction line is `<reactants> - -> <products> : <rate>` where a side is a list of
`<coefficient> <species>` pairs or the word NULL.  The result is the CSR network of include/rt.h
(reactant coefficients sigma_jk, net change v_k = products - reactants with zero entries dropped,
rate c_k), the initial counts, and the two run limits the file carries (`time` -> t_end, `steps`
-> max_firings; either may be absent).  Host-side text handling only: no arithmetic of the method.
"""
import math

import numpy as np


class ModelFileError(ValueError):
    pass


def _side(tokens, line_no):
    """[(species, coefficient)] of one side of a reaction."""
    if len(tokens) == 1 and tokens[0].upper() == "NULL":
        return []
    if not tokens or len(tokens) % 2:
        raise ModelFileError(f"line {line_no}: expected '<coefficient> <species>' pairs or NULL")
    out = []
    for c, name in zip(tokens[0::2], tokens[1::2]):
        try:
            coef = int(c)
        except ValueError:
            raise ModelFileError(f"line {line_no}: coefficient '{c}' is not an integer") from None
        if coef < 1:
            raise ModelFileError(f"line {line_no}: coefficient {coef} < 1")
        out.append((name, coef))
    return out


def parse_model(text):
    """Parse a model file.  Returns dict(net=..., x0=int64[N], species=[names], t_end=float (inf if
    no `time` line), max_firings=int (0 if no `steps` line))."""
    section = None
    counts, order, reactions = {}, [], []
    t_end, steps = math.inf, 0
    for line_no, raw in enumerate(text.splitlines(), 1):
        line = raw.split("//", 1)[0].strip()
        if not line:
            continue
        if line.startswith("#"):
            section = line[1:].strip().lower()
            if section not in ("init", "reactions", "end"):
                raise ModelFileError(f"line {line_no}: unknown section '# {section}'")
            continue
        if section == "init":
            name, sep, val = (s.strip() for s in line.partition("="))
            if not sep or not name or name in counts:
                raise ModelFileError(f"line {line_no}: expected '<species> = <count>' (once per species)")
            try:
                counts[name] = int(val)
            except ValueError:
                raise ModelFileError(f"line {line_no}: count '{val}' is not an integer") from None
            if counts[name] < 0:
                raise ModelFileError(f"line {line_no}: negative count")
            order.append(name)
        elif section == "reactions":
            body, sep, rate = line.rpartition(":")
            lhs, arrow, rhs = body.partition("- ->")
            if not sep or not arrow:
                raise ModelFileError(f"line {line_no}: expected '<reactants> - -> <products> : <rate>'")
            try:
                c = float(rate)
            except ValueError:
                raise ModelFileError(f"line {line_no}: rate '{rate.strip()}' is not a number") from None
            reactions.append((_side(lhs.split(), line_no), _side(rhs.split(), line_no), c, line_no))
        elif section == "end":
            name, sep, val = (s.strip() for s in line.partition("="))
            if name == "time" and sep:
                t_end = float(val)
            elif name == "steps" and sep:
                steps = int(val)
            else:
                raise ModelFileError(f"line {line_no}: expected 'time = <t>' or 'steps = <n>'")
        else:
            raise ModelFileError(f"line {line_no}: text before the first section")
    if not order or not reactions:
        raise ModelFileError("a model needs a '# init' and a '# reactions' section")
    index = {name: j for j, name in enumerate(order)}
    rp, rs, rg, sp, ss, sv, rate = [0], [], [], [0], [], [], []
    for lhs, rhs, c, line_no in reactions:
        react, change = {}, {}
        for side, sign in ((lhs, -1), (rhs, +1)):
            for name, coef in side:
                if name not in index:
                    raise ModelFileError(f"line {line_no}: species '{name}' has no initial count")
                j = index[name]
                change[j] = change.get(j, 0) + sign * coef
                if sign < 0:
                    react[j] = react.get(j, 0) + coef       # "1 A 1 A" means sigma = 2
        for j in sorted(react):
            rs.append(j)
            rg.append(react[j])
        rp.append(len(rs))
        for j in sorted(change):
            if change[j] != 0:
                ss.append(j)
                sv.append(change[j])
        sp.append(len(ss))
        rate.append(c)
    net = dict(n_species=len(order), n_reactions=len(reactions),
               react_ptr=np.asarray(rp, dtype=np.int64), react_species=np.asarray(rs, dtype=np.int32),
               react_sigma=np.asarray(rg, dtype=np.int32), stoich_ptr=np.asarray(sp, dtype=np.int64),
               stoich_species=np.asarray(ss, dtype=np.int32), stoich_v=np.asarray(sv, dtype=np.int32),
               rate=np.asarray(rate, dtype=np.float64))
    return dict(net=net, x0=np.asarray([counts[n] for n in order], dtype=np.int64), species=order,
                t_end=t_end, max_firings=steps)


def load_model(path):
    with open(path) as f:
        return parse_model(f.read())
