"""Independent restatement of one decoder-layer decode step from torch CPU library ops (fp64).

Used ONLY to pin the C oracle on cfg1 (SURVEY.md 8(c) "Whole layer: ... torch-CPU reference on cfg1
built from library ops (no shared code)").  It is vectorised differently from the oracle on
purpose: dense gathers, torch.softmax, complex-number RoPE.  Shares no code with oracle/ or the
CUDA library.
"""
import numpy as np
import torch


def bf16_bits_to_f64(u: np.ndarray) -> torch.Tensor:
    t = torch.from_numpy(np.ascontiguousarray(u).view(np.int16)).view(torch.bfloat16)
    return t.to(torch.float64)


def rope_complex(u: torch.Tensor, pos: torch.Tensor, base: float) -> torch.Tensor:
    """u [B, H, Dh]; rotate-half pairing (i, i+Dh/2) expressed as complex multiplication."""
    Dh = u.shape[-1]
    half = Dh // 2
    inv = torch.pow(torch.tensor(base, dtype=torch.float64), -torch.arange(half, dtype=torch.float64) * 2.0 / Dh)
    ang = pos.to(torch.float64)[:, None] * inv[None, :]                 # [B, half]
    z = torch.complex(u[..., :half], u[..., half:]) * torch.polar(torch.ones_like(ang), ang)[:, None, :]
    return torch.cat([z.real, z.imag], dim=-1)


def layer_step(shape, w, hidden, k_pool, v_pool, block_table, seq_lens):
    """Returns (out fp64 [B,d] before the final bf16 rounding, taps dict, k_pool', v_pool' bf16-bit arrays)."""
    W = {n: bf16_bits_to_f64(a) for n, a in w.items()}
    h = bf16_bits_to_f64(hidden)
    B, d = h.shape
    Hq, Hkv, Dh, page = shape.n_q_heads, shape.n_kv_heads, shape.head_dim, shape.page
    G = Hq // Hkv
    x = h * torch.rsqrt(h.pow(2).mean(-1, keepdim=True) + shape.rms_eps) * W["g1"]
    q = (x @ W["wq"].T).view(B, Hq, Dh)
    k = (x @ W["wk"].T).view(B, Hkv, Dh)
    v = (x @ W["wv"].T).view(B, Hkv, Dh)
    pos = torch.from_numpy(np.asarray(seq_lens, dtype=np.int64)) - 1
    q, k = rope_complex(q, pos, shape.rope_base), rope_complex(k, pos, shape.rope_base)
    kp = torch.from_numpy(k_pool.copy().view(np.int16)).view(torch.bfloat16)
    vp = torch.from_numpy(v_pool.copy().view(np.int16)).view(torch.bfloat16)
    bt = torch.from_numpy(np.asarray(block_table, dtype=np.int64))
    for b in range(B):
        p = int(pos[b])
        kp[bt[b, p // page], :, p % page, :] = k[b].to(torch.bfloat16)
        vp[bt[b, p // page], :, p % page, :] = v[b].to(torch.bfloat16)
    o = torch.zeros(B, Hq, Dh, dtype=torch.float64)
    for b in range(B):
        s = int(seq_lens[b])
        pages = bt[b, : (s + page - 1) // page]
        Kb = kp[pages].to(torch.float64).permute(1, 0, 2, 3).reshape(Hkv, -1, Dh)[:, :s]   # [Hkv, s, Dh]
        Vb = vp[pages].to(torch.float64).permute(1, 0, 2, 3).reshape(Hkv, -1, Dh)[:, :s]
        Kb = Kb.repeat_interleave(G, dim=0)                                               # [Hq, s, Dh]
        Vb = Vb.repeat_interleave(G, dim=0)
        sc = torch.einsum("hd,htd->ht", q[b], Kb) / np.sqrt(Dh)
        o[b] = torch.einsum("ht,htd->hd", torch.softmax(sc, dim=-1), Vb)
    h1 = h + o.reshape(B, Hq * Dh) @ W["wo"].T
    y = h1 * torch.rsqrt(h1.pow(2).mean(-1, keepdim=True) + shape.rms_eps) * W["g2"]
    a = torch.nn.functional.silu(y @ W["wgate"].T) * (y @ W["wup"].T)
    out = h1 + a @ W["wdown"].T
    taps = {"x": x, "q": q.reshape(B, -1), "k_new": k.reshape(B, -1), "v_new": v.reshape(B, -1),
            "o": o.reshape(B, -1), "h1": h1, "y": y, "a": a, "out": out}
    return out, taps, kp.view(torch.int16).numpy().view(np.uint16), vp.view(torch.int16).numpy().view(np.uint16)
