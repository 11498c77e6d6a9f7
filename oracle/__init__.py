"""CPU oracle for the Kara compress_window step — TEST INFRASTRUCTURE ONLY (see kara_oracle.h)."""
