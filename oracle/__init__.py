"""fp64 CPU oracle for the G-Core scoring hot path.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product path
(``paper_2507_22789_b200``) never imports it and shares no code with it.

See ``oracle/gcore_oracle.py`` for the functions and the passages they follow;
``oracle/balance_oracle.py`` holds the oracle of the repack + workload-balancing step,
``oracle/critic_oracle.py`` the oracle of the PPO critic path (value head, GAE, value loss),
``oracle/attention_oracle.py`` the oracle of the all-gather-KV distributed attention (sec 4.5).
"""
from .gcore_oracle import (  # noqa: F401
    AGG_TOKEN_MEAN,
    AGG_SEQ_MEAN,
    logits,
    token_logprobs,
    token_logprobs_row,
    group_filter,
    grpo_advantages,
    token_to_response,
    grpo_loss,
    grpo_loss_grad_logp,
    lm_head_backward,
    lm_head_backward_row,
    lm_head_backward_wrows,
    grpo_forward_backward,
)
from . import balance_oracle  # noqa: F401,E402
from . import critic_oracle  # noqa: F401,E402
from . import attention_oracle  # noqa: F401,E402
