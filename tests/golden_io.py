"""Reader for tests/golden/sh_closed_form.txt (text fixture; values cited from SURVEY.md §8(c))."""
import os

_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "sh_closed_form.txt")


def load():
    out = {"profile": {}, "cog": [], "psf_peak": None, "count": {}}
    with open(_PATH) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            t = line.split()
            if t[0] == "profile":
                out["profile"][tuple(int(x) for x in t[1:5])] = [float(x) for x in t[5:]]
            elif t[0] == "cog":
                out["cog"].append((tuple(int(x) for x in t[1:5]), float(t[5]), float(t[6])))
            elif t[0] == "psf_peak":
                out["psf_peak"] = (int(t[1]), int(t[2]), int(t[3]), float(t[4]))
            elif t[0] == "count":
                out["count"][t[1]] = {t[i]: int(t[i + 1]) for i in range(2, len(t), 2)}
    return out
