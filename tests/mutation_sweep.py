"""Mutation sweep of the CPU oracles (not collected by pytest; run by hand:  python tests/mutation_sweep.py [name | file ...]).

Every entry is ONE plausible mistake in oracle/*.py — a sign, an index, an operand order, a dropped term, a constant.  The script
copies oracle/ and tests/ to a temporary directory, applies one mutant at a time and runs the CPU suite there
(`pytest -m "not gpu"`; set MUT_ARGS='-k not(library)' to leave out the library-against-oracle comparisons and see the
independent pins alone).  A mutant that no test fails is printed as SURVIVED.  State at the end of round 2: 80 mutants,
78 killed; the two survivors are equivalent programs (clamping |r| at 480 instead of 448 before the nearest-code search
saturates to the same code; 1 / (amax / 448) against 448 / amax differs by an ulp on inputs the pins do not contain — the rule
itself is reading R42).  Nothing here is imported by the product or by a test."""
import os, shutil, subprocess, sys, tempfile
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
MUT = tempfile.mkdtemp(prefix="oracle_mutants_")
MUTANTS = [
 ("silu sign", "return z / (1.0 + torch.exp(-z))", "return z / (1.0 + torch.exp(z))"),
 ("gelu const", "0.044715 * z ** 3", "0.044715 * z ** 2"),
 ("gelu 0.5", "return 0.5 * z * (1.0 + torch.tanh(", "return 0.5 * z * (1.0 - torch.tanh("),
 ("swiglu operands", 'u = silu(linear(y, W[pre + "mlp.w1"], W[pre + "mlp.b1"])) * linear(y, W[pre + "mlp.w3"], W[pre + "mlp.b3"])', 'u = silu(linear(y, W[pre + "mlp.w3"], W[pre + "mlp.b3"])) * linear(y, W[pre + "mlp.w1"], W[pre + "mlp.b1"])'),
 ("ln eps outside", "return (x - mu) / torch.sqrt(var + eps)", "return (x - mu) / (torch.sqrt(var) + eps)"),
 ("modulate no 1+", "return layer_norm(x, eps) * (1.0 + scale) + shift", "return layer_norm(x, eps) * scale + shift"),
 ("modulate swap", "return layer_norm(x, eps) * (1.0 + scale) + shift", "return layer_norm(x, eps) * (1.0 + shift) + scale"),
 ("rms no gain", "return x / torch.sqrt(ms + eps) * g", "return x / torch.sqrt(ms + eps)"),
 ("rope freq", "omega = theta ** (-2.0 * j / d_a)", "omega = theta ** (-1.0 * j / d_a)"),
 ("rope sign", "out[..., 0::2] = a * c - b * s", "out[..., 0::2] = a * c + b * s"),
 ("rope halves", "a, b = x[..., 0::2], x[..., 1::2]", "a, b = x[..., :x.shape[-1] // 2], x[..., x.shape[-1] // 2:]"),
 ("token order", "return torch.stack([f.reshape(-1), h.reshape(-1), w.reshape(-1)], dim=1)", "return torch.stack([f.reshape(-1), w.reshape(-1), h.reshape(-1)], dim=1)"),
 ("attn scale", "scale = 1.0 / math.sqrt(d)", "scale = 1.0 / d"),
 ("lse", "lse[:, h] = (m + torch.log(z)).squeeze(-1)", "lse[:, h] = (torch.log(z)).squeeze(-1)"),
 ("merge weights", "w = torch.exp(L - m_safe)", "w = torch.exp(m_safe - L)"),
 ("shard size", "sz = -(-n // P)", "sz = n // P + 1"),
 ("patchify perm", "x = x.permute(1, 3, 5, 0, 2, 4, 6)                             # f' h' w' c i j k", "x = x.permute(1, 3, 5, 2, 4, 6, 0)"),
 ("unpatchify perm", "x = x.permute(3, 0, 4, 1, 5, 2, 6)                             # c f' i h' j w' k", "x = x.permute(3, 0, 4, 2, 6, 1, 5)"),
 ("tmlp silu pos", 'c = linear(silu(linear(_d(temb).reshape(1, -1), W["t_mlp.w1"], W["t_mlp.b1"])), W["t_mlp.w2"], W["t_mlp.b2"])', 'c = silu(linear(linear(_d(temb).reshape(1, -1), W["t_mlp.w1"], W["t_mlp.b1"]), W["t_mlp.w2"], W["t_mlp.b2"]))'),
 ("mod no silu", "    sc = silu(c)\n    mods", "    sc = c\n    mods"),
 ("mod order", "sh1, sc1, g1, sh2, sc2, g2 = mods[l]                                                      # step 2 order", "sc1, sh1, g1, sh2, sc2, g2 = mods[l]"),
 ("mod order 2", "sh1, sc1, g1, sh2, sc2, g2 = mods[l]                                                      # step 2 order", "sh1, sc1, g2, sh2, sc2, g1 = mods[l]"),
 ("joint order", "x = torch.cat([ctx, x], dim=0)                                                            # [ctx ; x] (R9)", "x = torch.cat([x, ctx], dim=0)"),
 ("cond pos", "pos = torch.cat([torch.zeros(Lc, 3, dtype=pos.dtype), pos], dim=0)                    # cond pos = 0 (R6)", "pos = torch.cat([torch.ones(Lc, 3, dtype=pos.dtype), pos], dim=0)"),
 ("attn resid no gate", 'x = x + g1 * linear(o, W[f"blocks.{l}.attn.wo"], W[f"blocks.{l}.attn.bo"])\n        if taps', 'x = x + linear(o, W[f"blocks.{l}.attn.wo"], W[f"blocks.{l}.attn.bo"])\n        if taps'),
 ("cross q no LN", 'qc = linear(layer_norm(x, eps), W[p + "wq"], W[p + "bq"]).reshape(-1, H, d)\n            kv = linear(ctx', 'qc = linear(x, W[p + "wq"], W[p + "bq"]).reshape(-1, H, d)\n            kv = linear(ctx'),
 ("cross no norm k", '            kc = rms_norm_heads(kc, _d(W[p + "gk"]), cfg["rms_eps"])\n            oc', '            oc'),
 ("final mod swap", "yf = modulate(xi, modf[0], modf[1], eps)", "yf = modulate(xi, modf[1], modf[0], eps)"),
 ("final rows", "xi = x[Lc:]                                                                                   # image tokens only", "xi = x[:x.shape[0] - Lc]"),
 ("dual txt/img weights", 'parts = (("txt", f"blocks.{l}.txt.", x[:Lc], m_txt), ("img", f"blocks.{l}.", x[Lc:], m_img))', 'parts = (("txt", f"blocks.{l}.", x[:Lc], m_txt), ("img", f"blocks.{l}.txt.", x[Lc:], m_img))'),
 ("dual mods swapped", 'parts = (("txt", f"blocks.{l}.txt.", x[:Lc], m_txt), ("img", f"blocks.{l}.", x[Lc:], m_img))', 'parts = (("txt", f"blocks.{l}.txt.", x[:Lc], m_img), ("img", f"blocks.{l}.", x[Lc:], m_txt))'),
 ("dual gate idx", "xa = xs + m[2] * linear(os_", "xa = xs + m[5] * linear(os_"),
 ("dual rope before cat", "outs.append(xa + m[5] * hm)", "outs.append(xa + m[2] * hm)"),
 ("euler sign", "x = x + (float(sigmas[i + 1]) - float(sigmas[i])) * v", "x = x + (float(sigmas[i]) - float(sigmas[i + 1])) * v"),
 ("guidance", "v = vu + float(guidance_scale) * (v - vu)", "v = v + float(guidance_scale) * (vu - v)"),
 ("block_rows gate", "return x + g2 * mlp(cfg, W, f\"blocks.{l}.\", y2)[1]", "return x + g1 * mlp(cfg, W, f\"blocks.{l}.\", y2)[1]"),
 ("block_rows resid", "x = x_in[rows] + g1 * linear(o", "x = x_in[rows] + g2 * linear(o"),
 ("txt mod silu", "    sc = silu(_d(c).reshape(1, -1))", "    sc = _d(c).reshape(1, -1)"),
 ("relayout", "return [full[a:b] for a, b in shard_bounds(full.shape[0], p_dst)]", "return [full[a:b] for a, b in shard_bounds(full.shape[0] - 1, p_dst)]"),
]
MORE = [
 ("oracle/fp8_oracle.py", "f8 bias", "v = 2.0 ** (e - 7) * (1.0 + m / 8.0)", "v = 2.0 ** (e - 8) * (1.0 + m / 8.0)"),
 ("oracle/fp8_oracle.py", "f8 subnormal", "v = 2.0 ** -6 * (m / 8.0)", "v = 2.0 ** -7 * (m / 8.0)"),
 ("oracle/fp8_oracle.py", "f8 nan", "if e == 15 and m == 7:", "if e == 15:"),
 ("oracle/fp8_oracle.py", "f8 ties", "((d_lo == d_hi) & (lo % 2 == 0))", "((d_lo == d_hi) & (lo % 2 == 1))"),
 ("oracle/fp8_oracle.py", "f8 sat", "a = r.double().abs().clamp(max=E4M3_MAX)", "a = r.double().abs().clamp(max=480.0)"),
 ("oracle/fp8_oracle.py", "f8 sign zero", "neg = (r < 0) | ((r == 0) & (torch.signbit(r)))", "neg = (r < 0)"),
 ("oracle/fp8_oracle.py", "f8 scale", "scale = torch.where(amax > 0, amax / m, torch.ones_like(amax))", "scale = torch.where(amax > 0, amax / 240.0, torch.ones_like(amax))"),
 ("oracle/fp8_oracle.py", "f8 inv", "inv = torch.where(amax > 0, m / amax, torch.ones_like(amax))", "inv = torch.where(amax > 0, 1.0 / (amax / m), torch.ones_like(amax))"),
 ("oracle/fp8_oracle.py", "f8 linear scales", "out = acc * a_scale.double()[:, None] * w_scale.double()[None, :]", "out = acc * a_scale.double()[:, None]"),
 ("oracle/mx_oracle.py", "mx offset", "sh = (e - 8).clamp(-127, 127)", "sh = (e - 7).clamp(-127, 127)"),
 ("oracle/mx_oracle.py", "mx clamp", "sh = (e - 8).clamp(-127, 127)", "sh = (e - 8).clamp(-126, 127)"),
 ("oracle/mx_oracle.py", "mx zero block", "return torch.where(a > 0, sh, torch.zeros_like(sh))", "return sh"),
 ("oracle/mx_oracle.py", "mx table", "t = torch.tensor([2.0 ** (c - 127) for c in range(255)]", "t = torch.tensor([2.0 ** (c - 128) for c in range(255)]"),
 ("oracle/mx_oracle.py", "mx block", "BLOCK = 32", "BLOCK = 16"),
 ("oracle/mx_oracle.py", "mx linear scale", "out += (a[:, b] @ w[:, b].T) * Xa[:, b][:, None] * Xw[:, b][None, :]", "out += (a[:, b] @ w[:, b].T) * Xa[:, b][:, None] * Xw[:, 0][None, :]"),
 ("oracle/mx_oracle.py", "mx amax", "sh = shared_exponent(v.abs().amax(dim=2))", "sh = shared_exponent(v.amax(dim=2).abs())"),
]
MORE += [
 ("oracle/sim_oracle.py", "sim srtf key", "r = min(cand, key=lambda q: ((requests[q][\"n_steps\"] - done[q]) * _cost(table, requests[q][\"shape_class\"], 1),", "r = max(cand, key=lambda q: ((requests[q][\"n_steps\"] - done[q]) * _cost(table, requests[q][\"shape_class\"], 1),"),
 ("oracle/sim_oracle.py", "sim edf key", "r = min(ready_set, key=lambda q: (requests[q][\"deadline_s\"], requests[q][\"arrival_s\"], q))", "r = min(ready_set, key=lambda q: (requests[q][\"arrival_s\"], requests[q][\"deadline_s\"], q))"),
 ("oracle/sim_oracle.py", "sim edf degree", "choice = cands[-1]", "choice = cands[0]"),
 ("oracle/sim_oracle.py", "sim edf slack", "if now + mig + (requests[r][\"n_steps\"] - done[r]) * _cost(table, c, p) <= requests[r][\"deadline_s\"]:", "if now + (requests[r][\"n_steps\"] - done[r]) * _cost(table, c, p) <= requests[r][\"deadline_s\"]:"),
 ("oracle/sim_oracle.py", "sim busy", "busy_s[r] += degree * dur", "busy_s[r] += dur"),
 ("oracle/sim_oracle.py", "sim fcfs pop", "r = queue[j].pop(0)", "r = queue[j].pop()"),
 ("oracle/sim_oracle.py", "sim p95", "p95_latency_s=lats[max(0, math.ceil(0.95 * len(lats)) - 1)] if lats else 0.0,", "p95_latency_s=lats[max(0, math.ceil(0.95 * len(lats)) - 2)] if lats else 0.0,"),
 ("oracle/sim_oracle.py", "sim failed", "failed = bool(timeout > 0 and lat > timeout)", "failed = bool(timeout > 0 and lat >= 0)"),
 ("oracle/sim_oracle.py", "sim mig count", "if mig > 0.0 or (last_set[r] is not None and last_set[r] != set_id):", "if mig > 0.0:"),
]
MORE += [
 ("oracle/dit_oracle.py", "rms eps outside", "return x / torch.sqrt(ms + eps) * g", "return x / (torch.sqrt(ms) + eps) * g"),
 ("oracle/dit_oracle.py", "rms sum", "ms = (x ** 2).mean(dim=-1, keepdim=True)", "ms = (x ** 2).sum(dim=-1, keepdim=True)"),
 ("oracle/dit_oracle.py", "ln unbiased", "var = ((x - mu) ** 2).mean(dim=-1, keepdim=True)", "var = ((x - mu) ** 2).sum(dim=-1, keepdim=True) / (x.shape[-1] - 1)"),
 ("oracle/dit_oracle.py", "linear transpose", "y = x @ _d(w).t()", "y = x @ _d(w)[:, :x.shape[-1]].t() if w.shape[0] != w.shape[1] else x @ _d(w)"),
 ("oracle/dit_oracle.py", "rope on v", "q, k = apply_rope(q, ang), apply_rope(k, ang)\n    if taps is not None:\n        taps[f\"b{l}.q\"]", "q, k, v = apply_rope(q, ang), apply_rope(k, ang), apply_rope(v, ang)\n    if taps is not None:\n        taps[f\"b{l}.q\"]"),
 ("oracle/dit_oracle.py", "softmax axis", "z = e.sum(dim=-1, keepdim=True)\n        p = e / z", "z = e.sum(dim=-1, keepdim=True)\n        p = e / e.sum(dim=0, keepdim=True)"),
 ("oracle/dit_oracle.py", "cross kv from x", "kv = linear(ctx, W[p + \"wkv\"], W[p + \"bkv\"])\n            kc, vc", "kv = linear(ctx * 1.0001, W[p + \"wkv\"], W[p + \"bkv\"])\n            kc, vc"),
 ("oracle/dit_oracle.py", "cross sign", "x = x + linear(oc.reshape(-1, D), W[p + \"wo\"], W[p + \"bo\"])\n            if taps", "x = x - linear(oc.reshape(-1, D), W[p + \"wo\"], W[p + \"bo\"])\n            if taps"),
 ("oracle/dit_oracle.py", "modf order", "modf = linear(sc, W[\"final.mod.w\"], W[\"final.mod.b\"]).reshape(2, -1)", "modf = linear(sc, W[\"final.mod.w\"], W[\"final.mod.b\"]).reshape(-1, 2).t()"),
 ("oracle/dit_oracle.py", "mods reshape", "mods = [linear(sc, W[f\"blocks.{l}.mod.w\"], W[f\"blocks.{l}.mod.b\"]).reshape(6, -1) for l in range(cfg[\"n_blocks\"])]", "mods = [linear(sc, W[f\"blocks.{l}.mod.w\"], W[f\"blocks.{l}.mod.b\"]).reshape(-1, 6).t() for l in range(cfg[\"n_blocks\"])]"),
 ("oracle/dit_oracle.py", "mlp second modulate", "y2 = modulate(x, sh2, sc2, eps)\n        u, hm = mlp(cfg, W, f\"blocks.{l}.\", y2)", "y2 = modulate(x, sh1, sc1, eps)\n        u, hm = mlp(cfg, W, f\"blocks.{l}.\", y2)"),
 ("oracle/dit_oracle.py", "qkv split", "q, k, v = (qkv[:, i * D:(i + 1) * D].reshape(T, H, d) for i in range(3))", "k, q, v = (qkv[:, i * D:(i + 1) * D].reshape(T, H, d) for i in range(3))"),
 ("oracle/dit_oracle.py", "heads layout", "q, k, v = (qkv[:, i * D:(i + 1) * D].reshape(T, H, d) for i in range(3))", "q, k, v = (qkv[:, i * D:(i + 1) * D].reshape(T, d, H).transpose(1, 2) for i in range(3))"),
 ("oracle/dit_oracle.py", "varlen shares temb", "return [dit_step(cfg, W, lat, te, co, split_p) for lat, te, co in zip(latents_list, temb_list, cond_list)]", "return [dit_step(cfg, W, lat, temb_list[0], co, split_p) for lat, te, co in zip(latents_list, temb_list, cond_list)]"),
 ("oracle/dit_oracle.py", "merge lse", "lse = m_safe + torch.log(z)                                    # log(0) = -inf when all shards are empty", "lse = m_safe + z"),
 ("oracle/dit_oracle.py", "dual qk gains", "k = rms_norm_heads(k, _d(W[pre + \"attn.gk\"]), cfg[\"rms_eps\"])\n        qs.append(q)", "k = rms_norm_heads(k, _d(W[pre + \"attn.gq\"]), cfg[\"rms_eps\"])\n        qs.append(q)"),
]
def setup():
    shutil.copytree(os.path.join(ROOT, "oracle"), os.path.join(MUT, "oracle"))
    shutil.copytree(os.path.join(ROOT, "tests"), os.path.join(MUT, "tests"))
    os.symlink(os.path.join(ROOT, "paper_2606_13501_b200"), os.path.join(MUT, "paper_2606_13501_b200"))
    for f in ("bench.py", "__graft_entry__.py", "BASELINE.json", "include", "MEASURED_PEAKS.json"):
        if os.path.exists(os.path.join(ROOT, f)):
            os.symlink(os.path.join(ROOT, f), os.path.join(MUT, f))
setup()
only = sys.argv[1:]
surv = []
ALL = [("oracle/dit_oracle.py",) + m for m in MUTANTS] + MORE
for fn, name, old, new in ALL:
    if only and name not in only and fn not in only: continue
    src = open(os.path.join(ROOT, fn)).read()
    if src.count(old) != 1:
        print(f"[skip] {name}: pattern occurs {src.count(old)} times"); continue
    for f2 in set(a[0] for a in ALL): shutil.copy(os.path.join(ROOT, f2), os.path.join(MUT, f2))
    open(os.path.join(MUT, fn), "w").write(src.replace(old, new))
    r = subprocess.run([sys.executable, "-m", "pytest", "tests", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider"] + os.environ.get("MUT_ARGS", "").split(), cwd=MUT, capture_output=True, text=True)
    killed = r.returncode != 0
    tail = [l for l in r.stdout.splitlines() if l.startswith("FAILED") or "passed" in l or "failed" in l][-2:]
    print(("killed " if killed else "SURVIVED ") + name, "|", " ".join(tail)[:160], flush=True)
    if not killed: surv.append(name)
print("survivors:", surv)
shutil.rmtree(MUT, ignore_errors=True)
