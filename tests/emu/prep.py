"""Rewrite CUDA launch syntax and dynamic smem declarations so a .cu file compiles as host C++."""
import re, sys

def match_back(s, i, open_c, close_c):
    # s[i] == close_c ; return index of matching open_c
    d = 0
    while i >= 0:
        if s[i] == close_c: d += 1
        elif s[i] == open_c:
            d -= 1
            if d == 0: return i
        i -= 1
    raise ValueError

def match_fwd(s, i, open_c, close_c):
    d = 0
    while i < len(s):
        if s[i] == open_c: d += 1
        elif s[i] == close_c:
            d -= 1
            if d == 0: return i
        i += 1
    raise ValueError

def split_top(a):
    out, d, cur = [], 0, ""
    for ch in a:
        if ch in "([{": d += 1
        if ch in ")]}": d -= 1
        if ch == "," and d == 0:
            out.append(cur.strip()); cur = ""
        else:
            cur += ch
    out.append(cur.strip())
    return out

def rewrite(s):
    # the asynchronous-copy wrappers (inline PTX) are replaced by the emulator's model of them
    s = s.replace('#include "fdas_tma.cuh"', '#include "emu_tma.h"')
    # the asynchronous-copy wrappers (inline PTX) are replaced by the emulator's model of them
    s = s.replace('#include "fdas_tma.cuh"', '#include "emu_tma.h"')
    s = re.sub(r"extern\s+__shared__\s+(?:__align__\(\d+\)\s+)?(\w+)\s+(\w+)\[\];", r"\1* \2 = (\1*)emu_dyn_smem();", s)
    while True:
        i = s.find("<<<")
        if i < 0: break
        j = i - 1
        while s[j].isspace(): j -= 1
        if s[j] == ">":
            j = match_back(s, j, "<", ">") - 1
        while j >= 0 and (s[j].isalnum() or s[j] == "_"): j -= 1
        k0 = j + 1
        kern = s[k0:i].strip()
        e = s.find(">>>", i)
        cfg = split_top(s[i + 3:e])
        while len(cfg) < 4: cfg.append("0")
        p0 = e + 3
        while s[p0].isspace(): p0 += 1
        assert s[p0] == "(", s[p0:p0+40]
        p1 = match_fwd(s, p0, "(", ")")
        args = s[p0 + 1:p1]
        name = kern.split("<")[0]
        rep = 'emu_launch(%s, %s, %s, "%s", [&]{ %s(%s); }, (cudaStream_t)(%s))' % (cfg[0], cfg[1], cfg[2], name, kern, args, cfg[3])
        s = s[:k0] + rep + s[p1 + 1:]
    return s

if __name__ == "__main__":
    open(sys.argv[2], "w").write(rewrite(open(sys.argv[1]).read()))
